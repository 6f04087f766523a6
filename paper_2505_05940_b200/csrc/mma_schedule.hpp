// mma_schedule.hpp -- host-side layout of the batched tensor-core vK kernel (vk_mma.cuh;
// DESIGN.md "Kernels / vk_mma").  No oracle code, no device code.
//
// Per time step and sample the kernel forms t[n][k] = sum_r H^n[k][r] q[r] (Eq. 9 in
// one pass, C eliminated by PAPER.md:283) as a GEMM  D[b][(n,k)] = Q[b][r] * Hs[(n,k)][r]^T  on
// tcgen05 tensor cores: M = 128 samples per tile, K = padded N_q, N = the (n,k) columns of a CTA.
// CTA (i,j) of the NGRP x NKB grid owns in-plane modes n of group i and the 16 rows k of block j.
// Operands are bf16 split hi + lo; three MMAs (hi*hi + lo*hi + hi*lo) per K chunk give ~2^-17
// relative accuracy, which the 1e-4 parity tolerance needs.
//
// Shared-memory operand layout (UMMA canonical K-major, no swizzle): a chunk of R rows x 16 K
// elements (bf16) is R*32 bytes; 8-row x 8-element core matrices of 128 contiguous bytes, the two
// K halves 128 B apart (LBO), 8-row groups 256 B apart (SBO).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace modal_host {

inline uint16_t bf16_rn(float x)
{
    uint32_t u; std::memcpy(&u, &x, 4);
    if ((u & 0x7f800000u) == 0x7f800000u) return (uint16_t)(u >> 16);   // inf / nan
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}
inline float bf16_to_float(uint16_t h) { uint32_t u = (uint32_t)h << 16; float f; std::memcpy(&f, &u, 4); return f; }

// byte offset of element (row r, k in 0..15) inside a canonical chunk
inline int umma_chunk_off(int r, int k) { return (r >> 3) * 256 + ((k >> 3) & 1) * 128 + (r & 7) * 16 + (k & 7) * 2; }

struct MmaLayout {
    int n_q = 0, n_phi = 0, KP = 0, KC = 0;     // padded K, K chunks of 16 (= k blocks of 16 rows)
    int NKB = 0, NGRP = 0, NG = 0, NC = 0;      // k blocks, n groups, modes per group, columns per CTA (NG*16)
    int NGP = 0;                                // NG padded to a multiple of 4 (float4 exchange rows)
    int G = 0;                                  // CTAs = NGRP * NKB
    size_t slab_bytes = 0;                      // per CTA: KC * 2 (hi, lo) * NC * 32
    std::vector<int> n0;                        // [NGRP+1] first in-plane mode of each group
};

// Returns false if the problem does not fit (grid of `sm` CTAs, `smem_limit` bytes each).
inline bool mma_layout(int n_q, int n_phi, int sm, size_t smem_limit, size_t smem_other, MmaLayout &L)
{
    L.n_q = n_q; L.n_phi = n_phi;
    L.KC = (n_q + 15) / 16; L.KP = L.KC * 16; L.NKB = L.KC;
    if (L.NKB > sm) return false;
    L.NGRP = std::min(n_phi, sm / L.NKB);
    L.NG = (n_phi + L.NGRP - 1) / L.NGRP;
    L.NGRP = (n_phi + L.NG - 1) / L.NG;
    L.NC = L.NG * 16;
    L.NGP = (L.NG + 3) / 4 * 4;
    L.G = L.NGRP * L.NKB;
    L.slab_bytes = (size_t)L.KC * 2 * L.NC * 32;
    if (L.NC > 256 || 2 * L.NC > 512) return false;
    if (L.slab_bytes + smem_other > smem_limit) return false;
    L.n0.resize(L.NGRP + 1);
    for (int i = 0; i <= L.NGRP; ++i) L.n0[i] = std::min(n_phi, i * L.NG);
    return true;
}

// Per-CTA operand slabs: [G][KC][2][NC*32 bytes]; CTA c = i * NKB + j.
template <class Get>   // Get(n,p,q) -> double (full symmetric H)
inline void pack_mma_slabs(const MmaLayout &L, Get get, std::vector<uint16_t> &slabs)
{
    slabs.assign((size_t)L.G * L.slab_bytes / 2, 0);
    for (int i = 0; i < L.NGRP; ++i)
        for (int j = 0; j < L.NKB; ++j) {
            uint16_t *base = &slabs[(size_t)(i * L.NKB + j) * L.slab_bytes / 2];
            for (int nl = 0; nl < L.NG; ++nl) {
                const int n = L.n0[i] + nl;
                if (n >= L.n0[i + 1]) break;
                for (int kk = 0; kk < 16; ++kk) {
                    const int k = j * 16 + kk;
                    if (k >= L.n_q) break;
                    const int row = nl * 16 + kk;
                    for (int r = 0; r < L.n_q; ++r) {
                        const float x = (float)get(n, k, r);
                        const uint16_t hi = bf16_rn(x), lo = bf16_rn(x - bf16_to_float(hi));
                        const size_t chunk = (size_t)(r >> 4) * 2 * L.NC * 32;
                        const int off = umma_chunk_off(row, r & 15);
                        base[(chunk + off) / 2] = hi;
                        base[(chunk + (size_t)L.NC * 32 + off) / 2] = lo;
                    }
                }
            }
        }
}

}  // namespace modal_host
