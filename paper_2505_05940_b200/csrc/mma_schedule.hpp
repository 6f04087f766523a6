// mma_schedule.hpp -- host-side layout of the batched tensor-core vK kernel (vk_mma.cuh;
// DESIGN.md "Kernels / vk_mma").  No oracle code, no device code.
//
// Per time step and sample the kernel forms t[n][k] = sum_r H^n[k][r] q[r] (Eq. 9 in
// one pass, C eliminated by PAPER.md:283) as a GEMM  D[b][(n,k)] = Q[b][r] * Hs[(n,k)][r]^T  on
// tcgen05 tensor cores: M = 128 samples per tile, K = padded N_q, N = the (n,k) columns of a CTA.
// CTA (i,j) of the NGRP x NKB grid owns in-plane modes n of group i and the RB rows k of block j
// (B-operand row = local mode * RB + local k).
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
    int n_q = 0, n_phi = 0, KP = 0, KC = 0;     // padded K, K chunks of 16
    int NKB = 0, RB = 0;                        // k blocks, rows k per block (multiple of 4, <= 32)
    int NGRP = 0, NG = 0, NC = 0;               // n groups, modes per group, operand columns per CTA (>= NG*RB, multiple of 16)
    int NG4 = 0;                                // float4 per partial-G row: ceil(NG / 4)
    int QS = 0;                                 // row stride (floats) of the q / partial-f exchange rows: max(KP, NKB*RB)
    int G = 0;                                  // CTAs = NGRP * NKB
    int nel_max = 0;                            // most (sample, k) elements one CTA owns per M tile
    size_t slab_bytes = 0;                      // per CTA: KC * 2 (hi, lo) * NC * 32
    std::vector<int> nlist;                     // [NGRP][NG] in-plane modes of each group (-1: empty slot)
    std::vector<int> klist, kcnt;               // [G][KC], [G]: the K chunks in which a CTA's slab holds a non-zero (pack_mma_slabs)
};

inline int mma_rows_owned_max(int NGRP) { return (128 + NGRP - 1) / NGRP; }

// One candidate shape; false if it does not fit.  smem_fixed = bytes besides the slab and the owner state.
// mode_class (optional, [n_phi]): modes of one group share a class.  For the sine-basis tensor the class is the index
// parity of the in-plane mode: H^n then couples a parity class of k only with one parity class of r, so most K chunks
// of a CTA's slab are zero and are skipped.
inline bool mma_layout_try(int n_q, int n_phi, int sm, size_t smem_limit, size_t smem_fixed, int NKB, int rb_align,
                           const std::vector<int> *mode_class, MmaLayout &L)
{
    L.n_q = n_q; L.n_phi = n_phi;
    L.KC = (n_q + 15) / 16; L.KP = L.KC * 16;
    L.NKB = NKB;
    L.RB = ((n_q + NKB - 1) / NKB + rb_align - 1) / rb_align * rb_align;
    if (L.RB > 32 || NKB > sm || L.KC > 64) return false;
    if (NKB > 1 && (NKB - 1) * L.RB >= n_q) return false;          // an empty k block
    const int max_groups = std::min(n_phi, sm / NKB);
    if (max_groups < 1) return false;
    std::vector<std::vector<int>> cls(4);
    for (int n = 0; n < n_phi; ++n) cls[mode_class ? ((*mode_class)[n] & 3) : 0].push_back(n);
    for (L.NG = (n_phi + max_groups - 1) / max_groups; L.NG <= 16; ++L.NG) {
        L.NGRP = 0;
        for (const auto &v : cls) L.NGRP += ((int)v.size() + L.NG - 1) / L.NG;
        if (L.NGRP <= max_groups) break;
    }
    L.NC = (L.NG * L.RB + 15) / 16 * 16;
    if (L.NG > 16 || L.NC > 256) return false;
    L.NG4 = (L.NG + 3) / 4;
    L.QS = std::max(L.KP, L.NKB * L.RB);
    L.G = L.NGRP * L.NKB;
    L.nel_max = mma_rows_owned_max(L.NGRP) * L.RB;
    L.slab_bytes = (size_t)L.KC * 2 * L.NC * 32;
    if (L.slab_bytes + smem_fixed + (size_t)2 * L.nel_max * (L.nel_max <= 512 ? 40 : 16) > smem_limit) return false;
    L.nlist.assign((size_t)L.NGRP * L.NG, -1);
    int g = 0;
    for (const auto &v : cls)
        for (size_t x = 0; x < v.size(); x += L.NG, ++g)
            for (int u = 0; u < L.NG && x + u < v.size(); ++u) L.nlist[(size_t)g * L.NG + u] = v[x + u];
    return true;
}

// Shape choice: the MMA time of a tile is ~ KC * 3 * NC / 2 cycles; the G hop reads NKB * NG4 rows per
// thread, the f hop NGRP partials per owned element.  force_nkb > 0 pins the number of k blocks
// (MODAL_MMA_NKB, tests / sweeps); rb_align = 16 keeps every tcgen05.ld column offset 16-aligned.
inline bool mma_layout(int n_q, int n_phi, int sm, size_t smem_limit, size_t smem_fixed, int force_nkb, int rb_align,
                       const std::vector<int> *mode_class, MmaLayout &L)
{
    double best = 1e300; bool found = false;
    const int KC = (n_q + 15) / 16;
    for (int NKB = 1; NKB <= std::min(4 * KC, sm); ++NKB) {
        if (force_nkb > 0 && NKB != force_nkb) continue;
        MmaLayout T;
        if (!mma_layout_try(n_q, n_phi, sm, smem_limit, smem_fixed, NKB, rb_align, mode_class, T)) continue;
        const double mma = (double)T.KC * 3.0 * T.NC / 2.0;
        const double ghop = T.NKB > 1 ? 600.0 + 40.0 * T.NKB * T.NG4 : 0.0;
        const double fhop = 600.0 + 12.0 * T.NGRP * ((T.nel_max + 127) / 128);
        const double cost = mma + ghop + fhop;
        if (cost < best) { best = cost; L = T; found = true; }
    }
    return found;
}

// Per-CTA operand slabs: [G][KC][2][NC*32 bytes]; CTA c = i * NKB + j; operand row = nl * RB + kk.  Also lists, per CTA,
// the K chunks whose slab part holds a non-zero (at least one entry, so that the accumulator is always written).
template <class Get>   // Get(n,p,q) -> double (full symmetric H)
inline void pack_mma_slabs(MmaLayout &L, Get get, std::vector<uint16_t> &slabs)
{
    slabs.assign((size_t)L.G * L.slab_bytes / 2, 0);
    L.klist.assign((size_t)L.G * L.KC, 0); L.kcnt.assign(L.G, 0);
    for (int i = 0; i < L.NGRP; ++i)
        for (int j = 0; j < L.NKB; ++j) {
            const int c = i * L.NKB + j;
            uint16_t *base = &slabs[(size_t)c * L.slab_bytes / 2];
            std::vector<char> used(L.KC, 0);
            for (int nl = 0; nl < L.NG; ++nl) {
                const int n = L.nlist[(size_t)i * L.NG + nl];
                if (n < 0) continue;
                for (int kk = 0; kk < L.RB; ++kk) {
                    const int k = j * L.RB + kk;
                    if (k >= L.n_q) break;
                    const int row = nl * L.RB + kk;
                    for (int r = 0; r < L.n_q; ++r) {
                        const float x = (float)get(n, k, r);
                        if (x == 0.f) continue;
                        used[r >> 4] = 1;
                        const uint16_t hi = bf16_rn(x), lo = bf16_rn(x - bf16_to_float(hi));
                        const size_t chunk = (size_t)(r >> 4) * 2 * L.NC * 32;
                        const int off = umma_chunk_off(row, r & 15);
                        base[(chunk + off) / 2] = hi;
                        base[(chunk + (size_t)L.NC * 32 + off) / 2] = lo;
                    }
                }
            }
            int cnt = 0;
            for (int kc = 0; kc < L.KC; ++kc) if (used[kc]) L.klist[(size_t)c * L.KC + cnt++] = kc;
            if (!cnt) { L.klist[(size_t)c * L.KC] = 0; cnt = 1; }
            L.kcnt[c] = cnt;
        }
}

}  // namespace modal_host
