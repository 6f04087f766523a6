// mma_schedule.hpp -- host-side layout of the batched tensor-core vK kernel (vk_mma.cuh;
// DESIGN.md "Kernels / vk_mma").  No oracle code, no device code.
//
// Per time step and sample the kernel forms t[n][k] = sum_r H^n[k][r] q[r] (Eq. 9 in
// one pass, C eliminated by PAPER.md:283) as a GEMM  D[b][(n,k)] = Q[b][r] * Hs[(n,k)][r]^T  on
// tcgen05 tensor cores: M = 128 samples per tile, K = the transverse modes r, N = the (n,k) columns of a CTA.
// CTA (i,j) of the NGRP x NKB grid owns the in-plane modes n of group i and the rows k of block j.
// Operands are bf16 split hi + lo; three MMAs (hi*hi + lo*hi + hi*lo) per K chunk give ~2^-17
// relative accuracy, which the 1e-4 parity tolerance needs.
//
// Operand order of the transverse modes.  The k blocks are contiguous ranges of the plan's INTERNAL mode
// order, aligned to its classes (for the sine-basis plate: the four index parities); every
// block starts on a 16-element boundary of the operand K axis (koff), so a K chunk of 16 never straddles two
// blocks.  H^n couples a parity class of k with ONE parity class of r, so a CTA's slab is non-zero in only a few K
// chunks; the host lists them per CTA from the actual non-zeros of H (an uploaded dense H simply lists them all).
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

constexpr int MMA_RB_MAX = 56;      // most rows k of one block (the epilogue keeps a sample's block of q in registers)
constexpr int MMA_NG_MAX = 8;       // most in-plane modes of one group
constexpr int MMA_KCL_MAX = 64;     // most K chunks one CTA multiplies
constexpr int MMA_FBLK_MAX = 16;    // most k blocks whose owners a CTA waits for
constexpr int MMA_MT_MAX = 8;       // most M tiles (of 128 samples) of one launch

struct MmaBlock { int k0, nb, koff; };            // first internal mode, modes, offset on the operand K axis (multiple of 16)

struct MmaLayout {
    int n_q = 0, n_phi = 0;
    int NKB = 0;                                // k blocks
    std::vector<MmaBlock> blocks;
    int RBT = 0;                                // TMEM columns per in-plane mode: 32 or 64 (>= the largest block)
    int RBQ = 0;                                // quads (4 consecutive k) per block in the exchange rows: ceil(max nb / 4)
    int KP = 0, KC = 0;                         // operand K extent (sum of the padded blocks), chunks of 16
    int NGRP = 0, NG = 0, NG4 = 0;              // n groups, most modes per group, float4 per partial-G row
    std::vector<int> nlist;                     // [NGRP][NG] in-plane modes of each group (-1: empty slot)
    int NC = 0;                                 // TMEM columns of one accumulator slot = NG * RBT (multiple of 16, <= 256)
    int S = 0;                                  // accumulator slots in TMEM: min(3, 512 / NC); 2 in cluster mode
    int CL = 0;                                 // 1: the NKB CTAs of a group form a thread-block cluster (partial G through distributed shared memory)
    int G = 0;                                  // CTAs = NGRP * NKB
    int rows_max = 0;                           // most sample rows of a tile one CTA owns for the update
    int KCL = 0;                                // most K chunks of any CTA (slab size)
    size_t slab_bytes = 0;                      // per CTA: KCL * 2 (hi, lo) * NC * 32
    std::vector<int> klist, kcnt;               // [G][KCL], [G]: global K chunks in which a CTA's slab holds a non-zero
    std::vector<int> fblk, fcnt;                // [G][MMA_FBLK_MAX], [G]: k blocks whose owners publish what the CTA reads (own block first)
    double cost = 0;
};

inline int mma_rows_owned_max(int NGRP) { return (128 + NGRP - 1) / NGRP; }

// k blocks: every class (contiguous range of the internal order; class_start has ncls+1 entries) cut into
// `split` nearly equal parts, more if a part would exceed MMA_RB_MAX.
inline void mma_blocks(const std::vector<int> &class_start, int split, std::vector<MmaBlock> &blocks)
{
    blocks.clear();
    int koff = 0;
    for (size_t c = 0; c + 1 < class_start.size(); ++c) {
        const int k0 = class_start[c], len = class_start[c + 1] - k0;
        if (len <= 0) continue;
        int parts = std::max(split, (len + MMA_RB_MAX - 1) / MMA_RB_MAX);
        parts = std::min(parts, len);
        for (int p = 0; p < parts; ++p) {
            const int a = k0 + (int)((long long)len * p / parts), b = k0 + (int)((long long)len * (p + 1) / parts);
            blocks.push_back({a, b - a, koff});
            koff += (b - a + 15) / 16 * 16;
        }
    }
}

// One candidate shape: blocks given, NG modes per group.  mode_class [n_phi]: modes of one group share a class.
// `nz(n, k_int, r_int)` tells whether H^n[k][r] is non-zero.  Returns false if the shape does not fit the machine.
// cluster_cap[s] (s = 2, 4, 8): thread-block clusters of s CTAs the device keeps co-resident with this kernel (0: none).
template <class NZ>
inline bool mma_layout_try(int n_q, int n_phi, int sm, size_t smem_limit, size_t smem_fixed, const std::vector<MmaBlock> &blocks,
                           int NG, const std::vector<int> &mode_class, NZ nz, const int *cluster_cap, MmaLayout &L)
{
    L = MmaLayout();
    L.n_q = n_q; L.n_phi = n_phi; L.blocks = blocks; L.NKB = (int)blocks.size();
    if (L.NKB < 1 || L.NKB > MMA_FBLK_MAX - 1 || NG < 1 || NG > MMA_NG_MAX) return false;
    int nbmax = 0;
    for (const MmaBlock &b : blocks) nbmax = std::max(nbmax, b.nb);
    if (nbmax > MMA_RB_MAX) return false;
    L.RBT = nbmax <= 32 ? 32 : 64; L.RBQ = (nbmax + 3) / 4;      // the epilogue reads the accumulator in units of 32 columns
    L.KP = blocks.back().koff + (blocks.back().nb + 15) / 16 * 16; L.KC = L.KP / 16;
    std::vector<std::vector<int>> cls(4);
    for (int n = 0; n < n_phi; ++n) cls[mode_class[n] & 3].push_back(n);
    L.NG = NG; L.NG4 = (NG + 3) / 4;
    L.NGRP = 0;
    for (const auto &v : cls) L.NGRP += ((int)v.size() + NG - 1) / NG;
    L.G = L.NGRP * L.NKB;
    if (L.G > sm || L.NGRP > 128) return false;
    L.NC = NG * L.RBT;
    if (L.NC > 256) return false;
    L.S = std::min(3, 512 / L.NC);
    L.CL = (L.NKB == 2 || L.NKB == 4 || L.NKB == 8) && cluster_cap && cluster_cap[L.NKB] >= L.NGRP;
    if (L.CL) L.S = std::min(L.S, 2);
    L.rows_max = mma_rows_owned_max(L.NGRP);
    L.nlist.assign((size_t)L.NGRP * NG, -1);
    {   // groups: the modes of a class spread evenly over its groups (balanced MMA work)
        int g = 0;
        for (const auto &v : cls) {
            const int ng = ((int)v.size() + NG - 1) / NG;
            for (int x = 0; x < ng; ++x) {
                const int a = (int)((long long)v.size() * x / ng), b = (int)((long long)v.size() * (x + 1) / ng);
                for (int u = a; u < b; ++u) L.nlist[(size_t)(g + x) * NG + (u - a)] = v[u];
            }
            g += ng;
        }
    }
    // K chunks and source blocks of every CTA from the non-zeros of its part of H
    const int KC = L.KC;
    std::vector<int> chunk_block(KC, 0);
    for (int j = 0; j < L.NKB; ++j)
        for (int kc = blocks[j].koff / 16; kc < (blocks[j].koff + blocks[j].nb + 15) / 16; ++kc) chunk_block[kc] = j;
    std::vector<std::vector<int>> lists(L.G);
    L.KCL = 1;
    for (int i = 0; i < L.NGRP; ++i)
        for (int j = 0; j < L.NKB; ++j) {
            std::vector<char> used(KC, 0);
            for (int nl = 0; nl < NG; ++nl) {
                const int n = L.nlist[(size_t)i * NG + nl];
                if (n < 0) continue;
                for (int kk = 0; kk < blocks[j].nb; ++kk)
                    for (int jr = 0; jr < L.NKB; ++jr)
                        for (int rr = 0; rr < blocks[jr].nb; ++rr)
                            if (!used[(blocks[jr].koff + rr) >> 4] && nz(n, blocks[j].k0 + kk, blocks[jr].k0 + rr))
                                used[(blocks[jr].koff + rr) >> 4] = 1;
            }
            std::vector<int> &l = lists[(size_t)i * L.NKB + j];
            for (int kc = 0; kc < KC; ++kc) if (used[kc]) l.push_back(kc);
            if (l.empty()) l.push_back(blocks[j].koff / 16);     // at least one chunk, so that the accumulator is always written
            L.KCL = std::max(L.KCL, (int)l.size());
        }
    if (L.KCL > MMA_KCL_MAX) return false;
    L.slab_bytes = (size_t)L.KCL * 2 * L.NC * 32;
    const size_t own = (size_t)2 * L.rows_max * L.RBQ * 4 * 44;                    // fp64 (q, v, kv, kq, r) + fp32 w of the owned elements: at least two tiles per launch
    if (L.slab_bytes + smem_fixed + own + (size_t)std::max(2, L.KCL) * 8192 > smem_limit) return false;   // ring: at least one tile's chunks
    L.klist.assign((size_t)L.G * L.KCL, 0); L.kcnt.assign(L.G, 0);
    L.fblk.assign((size_t)L.G * MMA_FBLK_MAX, 0); L.fcnt.assign(L.G, 0);
    for (int c = 0; c < L.G; ++c) {
        const std::vector<int> &l = lists[c];
        L.kcnt[c] = (int)l.size();
        for (size_t x = 0; x < l.size(); ++x) L.klist[(size_t)c * L.KCL + x] = l[x];
        int *fb = &L.fblk[(size_t)c * MMA_FBLK_MAX];
        int cnt = 0;
        fb[cnt++] = c % L.NKB;                                   // own block: the epilogue reads this sample's q over it
        for (int kc : l) {
            const int jb = chunk_block[kc];
            bool seen = false;
            for (int x = 0; x < cnt; ++x) seen |= fb[x] == jb;
            if (!seen) fb[cnt++] = jb;
        }
        L.fcnt[c] = cnt;
    }
    // rough cost of one tile-step in SM cycles (per CTA): MMA issue, L2 bytes at ~32 B/clk/SM, owner gather (16 strong
    // loads in flight per lane, 64 lanes per team) and a latency term for the hops
    const double mma = (double)L.KCL * 3.0 * L.NC / 2.0;
    const double bytes = (double)L.KCL * 8192 + 128.0 * L.RBQ * 16 * 2 + (double)L.NGRP * L.rows_max * L.RBQ * 16 + 128.0 * L.NG4 * 16 * L.NKB;
    const double gather = 700.0 * std::ceil((double)L.NGRP * L.rows_max * L.RBQ / (16.0 * 64.0));
    const double idle = (double)(sm - L.G) / sm;
    const double ghop = L.NKB == 1 ? 0.0 : L.CL ? 800.0 : 4500.0;          // partial-G exchange: distributed shared memory vs polling through L2
    L.cost = (std::max(mma, bytes / 32.0) + gather + ghop + 30.0 * L.NGRP) * (1.0 + idle);
    return true;
}

// Shape choice over the class splits and group sizes.  force_split / force_ng > 0 pin them (plan options, tests / sweeps).
template <class NZ>
inline bool mma_layout(int n_q, int n_phi, int sm, size_t smem_limit, size_t smem_fixed, const std::vector<int> &class_start,
                       const std::vector<int> &mode_class, NZ nz, int force_split, int force_ng, const int *cluster_cap, MmaLayout &L)
{
    bool found = false;
    for (int split = 1; split <= 4; ++split) {
        if (force_split > 0 && split != force_split) continue;
        std::vector<MmaBlock> blocks;
        mma_blocks(class_start, split, blocks);
        for (int NG = 1; NG <= MMA_NG_MAX; ++NG) {
            if (force_ng > 0 && NG != force_ng) continue;
            MmaLayout T;
            if (!mma_layout_try(n_q, n_phi, sm, smem_limit, smem_fixed, blocks, NG, mode_class, nz, cluster_cap, T)) continue;
            if (!found || T.cost < L.cost) { L = T; found = true; }
        }
    }
    return found;
}

// Per-CTA operand slabs: [G][KCL][2][NC*32 bytes], chunk x of the CTA's list at x * 2 * NC * 32 (hi, then lo at + NC*32);
// operand row = nl * RBT + kk.  get(n, k_int, r_int) -> double (full symmetric H in internal order).
template <class Get>
inline void pack_mma_slabs(const MmaLayout &L, Get get, std::vector<uint16_t> &slabs)
{
    slabs.assign((size_t)L.G * L.slab_bytes / 2, 0);
    std::vector<int> kop(L.KP, -1);                               // operand K position -> internal mode
    for (const MmaBlock &b : L.blocks) for (int x = 0; x < b.nb; ++x) kop[b.koff + x] = b.k0 + x;
    for (int i = 0; i < L.NGRP; ++i)
        for (int j = 0; j < L.NKB; ++j) {
            const int c = i * L.NKB + j;
            uint16_t *base = &slabs[(size_t)c * L.slab_bytes / 2];
            for (int x = 0; x < L.kcnt[c]; ++x) {
                const int kc = L.klist[(size_t)c * L.KCL + x];
                const size_t chunk = (size_t)x * 2 * L.NC * 32;
                for (int nl = 0; nl < L.NG; ++nl) {
                    const int n = L.nlist[(size_t)i * L.NG + nl];
                    if (n < 0) continue;
                    for (int kk = 0; kk < L.blocks[j].nb; ++kk) {
                        const int row = nl * L.RBT + kk;
                        for (int e = 0; e < 16; ++e) {
                            const int r = kop[kc * 16 + e];
                            if (r < 0) continue;
                            const float v = (float)get(n, L.blocks[j].k0 + kk, r);
                            if (v == 0.f) continue;
                            const uint16_t hi = bf16_rn(v), lo = bf16_rn(v - bf16_to_float(hi));
                            const int off = umma_chunk_off(row, e);
                            base[(chunk + off) / 2] = hi;
                            base[(chunk + (size_t)L.NC * 32 + off) / 2] = lo;
                        }
                    }
                }
            }
        }
}

}  // namespace modal_host
