// vk_stream.cuh -- STREAMING tensor-core von Karman kernel: batches of 8..64 samples on a tensor too large to keep in shared memory
// (C4: N_q = 400, N_phi = 200; SURVEY.md 8(a) rows a2-a6, 8(d) "C4 b16 / b64").  Layout: stream_schedule.hpp.  DESIGN.md "vk_stream".
//
// Per step (Eq. 9 with C eliminated; update PAPER.md:120-124 Eq. 10 in delta form, R4):
//   t[(n,k)][b] = sum_r H^n[k][r] q[b][r]          tcgen05.mma, M = 128 rows k of one (mode n, k block) tile, N = NB samples, K = r;
//                                                  H streamed from L2 by TMA as bf16 hi + lo (one bulk copy per tile into a ring of tile-sized
//                                                  stages), q rebuilt in shared memory as bf16 hi + lo; per K chunk three MMAs (hi*hi + lo*hi +
//                                                  hi*lo) at NB = 64, two at NB <= 32 (H_hi * [q_hi ; q_lo] with N = 2 NB, then H_lo * q_hi: the
//                                                  epilogues add the two column halves); fp32 accumulators of ALL tiles of the CTA in TMEM
//   G_n[b] = sum_k q[b][k] t[(n,k)][b]             epilogue 1: thread <-> row k; products reduced over the 128 rows by a butterfly that leaves
//                                                  each lane with one sample, partial G per k block exchanged through L2 (tagged words)
//   f[b][k] = sum_n s_n[b] G_n[b] t[(n,k)][b]      epilogue 2: the thread's row accumulates over the CTA's tiles in registers
//   owners: gather the partial f of their rows from the CTAs of the block, fp64 update, publish q^{n+1} (tagged fp32), pickup partials.
//
// Warps: 0 = P (TMA producer of the H stream), 1 = M (MMA issue), 2 = W (pickup: out[b][n], one sample per CTA), 4-7 = E (epilogues),
// 8-15 = O (owners).  Every exchange is one-way through L2 with the step's 2-bit tag in the low mantissa bits of each fp32 word.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_mma.cuh"   // tcgen05 / mbarrier / tagged-word helpers

namespace modal_dev {

constexpr int ST_THREADS = 512;
constexpr int ST_BCH_MAX_DEV = 16, ST_TILES_MAX_DEV = 16, ST_NKB_MAX_DEV = 8, ST_SENT_MAX_DEV = 256, ST_CTA_STRIDE = 6 + ST_BCH_MAX_DEV + 1 + ST_SENT_MAX_DEV;
constexpr unsigned ST_POLL_SLEEP = 100;   // ns between polling rounds
constexpr int SB_FULL = 0, SB_EMPTY = 16, SB_ACCF = 32, SB_ACCE = 48, SB_BRDY = 49, SB_FDONE = 50, SB_TPTR = 56, SB_ABORT = 57;
constexpr int ST_BARS_BYTES = 512;
constexpr int ST_NSTG_MAX = 8;          // ring stages (one tile each)

struct StreamArgs {
    const uint16_t *A;          // H stream: per tile its K chunks, 8 KiB each (hi 4 KiB, lo 4 KiB), UMMA canonical K-major
    const int *cta_tab, *tile_tab; int tile_stride;
    const int *blk;             // [NKB][4]: k0, nb, koff, first CTA of the block
    const int *blk_nctas;       // [NKB]
    int NKB, KOP, G, NSTG, rows_max, bch_max, LPQ;
    int stage_bytes;            // ring stage = the most K chunks of a tile x 8 KiB
    int n_q, n_phi, NQP, batch, n_steps;
    int coeff_stride_q, coeff_stride_phi;
    const double *kv, *kq, *r, *astart;
    const float *s, *w;
    const double *q0, *v0;
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; const int *kperm; int *first_bad;
    uint32_t *qx;               // [NB][KOP]            q, tagged fp32, operand order
    uint32_t *Gx;               // [n_phi][NKB][NB]     partial G per k block, tagged
    uint32_t *fx;               // [G][128][NB]         partial f per CTA, tagged
    unsigned long long *px;     // [4][G][NB][2]        pickup partials {o, epoch}, {|q|^2, epoch}
    uint32_t *wflag;            // [NB]                 steps of sample b the pickup warp has written out
    int *timeout_flag;
    long long *timing;          // optional [G][16]
};

struct StreamSmem { size_t bars, tab, ss, wsum, seta, sq, sv, coef, pk, misc, bop, ring, total; };
__host__ __device__ inline StreamSmem stream_smem_layout(int NB, int rows_max, int bch_max, int tile_stride, int nstg, int stage_bytes)
{
    StreamSmem L; size_t o = 0;
    const size_t nel = (size_t)rows_max * NB;
    L.bars = o;  o += ST_BARS_BYTES;
    L.tab = o;   o += (size_t)(ST_CTA_STRIDE + ST_TILES_MAX_DEV * tile_stride + 4 * ST_NKB_MAX_DEV + ST_NKB_MAX_DEV) * 4;
    o = flow_align(o, 16);
    L.ss = o;    o += (size_t)ST_TILES_MAX_DEV * NB * 4;       // s_n[b] of the CTA's tiles
    L.wsum = o;  o += (size_t)2 * 4 * NB * 4;                  // per-warp partial G, by tile parity
    L.seta = o;  o += (size_t)ST_TILES_MAX_DEV * NB * 4;       // eta[tile][b]
    L.sq = o;    o += nel * 8;
    L.sv = o;    o += nel * 8;
    L.coef = o;  o += nel * 28;                                // kv, kq, r fp64 + w fp32
    L.pk = o;    o += nel * 8 * 2;                             // pickup partials [step parity][row][b] float2
    L.misc = o;  o += 16;                                      // sbad, wdone
    o = flow_align(o, 128);
    L.bop = o;   o += (size_t)bch_max * NB * 64;               // q operand chunks: [slot][hi NB x 16 | lo NB x 16] bf16
    o = flow_align(o, 128);
    L.ring = o;  o += (size_t)nstg * stage_bytes;
    L.total = o;
    return L;
}

// Sum over the 32 lanes of a warp of v[c] for every column c of the unit, by halving exchanges: afterwards the lane holds the
// total of column `col` (U = 32: one column per lane; U = 16: lane pairs hold the same column).
template <int U>
__device__ __forceinline__ float warp_reduce_scatter(float (&v)[U], const int lane, int &col)
{
    col = 0;
    int m = 16;
#pragma unroll
    for (int half = U / 2; half >= 1; half >>= 1, m >>= 1) {
        const bool up = (lane & m) != 0;
#pragma unroll
        for (int i = 0; i < half; ++i) {
            const float send = up ? v[i] : v[i + half];
            const float keep = up ? v[i + half] : v[i];
            v[i] = keep + __shfl_xor_sync(FLOW_FULL, send, m);
        }
        if (up) col += half;
    }
    if (U == 16) v[0] += __shfl_xor_sync(FLOW_FULL, v[0], 1);
    return v[0];
}

__device__ __forceinline__ uint32_t ld_relaxed1(const uint32_t *p)
{
    uint32_t w;
    asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(w) : "l"(p) : "memory");
    return w;
}
__device__ __forceinline__ void st_relaxed1(uint32_t *p, uint32_t w)
{
    asm volatile("st.relaxed.gpu.global.b32 [%0], %1;" ::"l"(p), "r"(w) : "memory");
}
// one non-blocking probe of a phase
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// one try_wait on the fast path; the bounded loop only when the phase is not complete yet
__device__ __forceinline__ void mbar_wait_fast(uint32_t bar, uint32_t parity, volatile int *abortp)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (!ok) mbar_wait(bar, parity, abortp);
}
__device__ __forceinline__ bool elect_one_sync()
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
// One warp waits for the tag on a list of single words (sentinels), four per lane and round, sleeping between rounds.  Everybody else
// sleeps on a CTA barrier meanwhile: 19 k threads spinning on L2 with eight loads each slow every store and hop of the step tenfold.
template <class Addr>
__device__ __forceinline__ void warp_poll_sentinels(const int count, const int lane, const uint32_t tag, volatile int *s_abort, Addr addr)
{
    for (int s0 = 0; s0 < count; s0 += 128) {
        const uint32_t *ptr[4];
        unsigned pend = 0, spins = 0;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int x = s0 + 32 * u + lane;
            ptr[u] = nullptr;
            if (x < count) { ptr[u] = addr(x); if (ptr[u]) pend |= 1u << u; }
        }
        while (pend) {
            uint32_t v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) if (pend >> u & 1) v[u] = ld_relaxed1(ptr[u]);
#pragma unroll
            for (int u = 0; u < 4; ++u) if ((pend >> u & 1) && (v[u] & 3u) == tag) pend &= ~(1u << u);
            if (pend) {
                if ((++spins & 255u) == 0 && (*s_abort || spins > (1u << 22))) { *s_abort = 1; break; }
                __nanosleep(ST_POLL_SLEEP);
            }
        }
    }
    __syncwarp();
}
template <int U> struct TmemUnit;
template <> struct TmemUnit<32> { static __device__ __forceinline__ void ld(uint32_t t, uint32_t (&u)[32]) { tmem_ld32_nowait(t, u); } };
template <> struct TmemUnit<16> { static __device__ __forceinline__ void ld(uint32_t t, uint32_t (&u)[16]) { tmem_ld16_nowait(t, u); } };

// CTA-uniform view
struct StreamCta {
    int c, jb, x;               // CTA, its k block, its index among the block's CTAs
    int tile0, ntiles, nbch, row0, rows;
    int k0, nb, koff, cta0, nct;
    uint64_t *bars;
    const int *ctab, *ttab, *blk, *bnct;
    volatile int *s_abort;
    float *ss, *wsum, *seta; float2 *pk;
    double *sq, *sv; unsigned char *coef;
    int *sbad; volatile int *wdone;
    unsigned char *bop, *ring;
    uint32_t tbase;
    size_t nel;
};

// DUAL (NB <= 32): a tile's accumulator has 2 NB columns -- [0, NB) = H_hi q_hi + H_lo q_hi, [NB, 2 NB) = H_hi q_lo -- so that the two MMAs
// that use H_hi (against q_hi and q_lo) are ONE instruction with the B operand [q_hi ; q_lo] of 2 NB rows (the two halves are adjacent
// in the operand layout): two MMAs and 8 KiB of shared-memory operand reads per K chunk instead of three and 12 KiB.  The epilogues
// add the halves.  At NB = 64 the tiles of a CTA would not fit the 512 TMEM columns, so the three-MMA form stays.
template <int NB> struct StreamDual { static constexpr bool value = NB <= 32; static constexpr int TSTR = NB <= 32 ? 2 * NB : NB; };
template <int NB, int U, int NU>
__device__ __forceinline__ void stream_load_t(const uint32_t lane_addr, const int i, uint32_t (&tu)[NU][U])
{
    constexpr int TSTR = StreamDual<NB>::TSTR;
    if (StreamDual<NB>::value) {
        uint32_t lo[NU][U];
#pragma unroll
        for (int u = 0; u < NU; ++u) {
            TmemUnit<U>::ld(lane_addr + (uint32_t)(i * TSTR + u * U), tu[u]);
            TmemUnit<U>::ld(lane_addr + (uint32_t)(i * TSTR + NB + u * U), lo[u]);
        }
        tmem_ld_wait();
#pragma unroll
        for (int u = 0; u < NU; ++u)
#pragma unroll
            for (int c = 0; c < U; ++c) tu[u][c] = __float_as_uint(__uint_as_float(tu[u][c]) + __uint_as_float(lo[u][c]));
    } else {
#pragma unroll
        for (int u = 0; u < NU; ++u) TmemUnit<U>::ld(lane_addr + (uint32_t)(i * TSTR + u * U), tu[u]);
        tmem_ld_wait();
    }
}

// q^n of the CTA's K chunks -> bf16 hi / lo operand chunks in shared memory (the B operand of the step's MMAs), by the 128 epilogue
// threads and the 256 owner threads together (the owners are idle between publishing q^n and the forces of step n).
constexpr int ST_BUILDERS = 384;
template <int NB, int IF>   // IF: items (two 16-byte loads each) a thread keeps in flight
__device__ __forceinline__ void stream_build_B(const StreamArgs &a, const StreamCta &C, const int first, const uint32_t tag)
{
    // item = (chunk slot, half of its 16 K, sample): 8 consecutive k of one sample = one 16-byte row of a core matrix;
    // four items per round: their eight 16-byte loads are in flight together
    for (int idx0 = first; idx0 < C.nbch * 2 * NB; idx0 += IF * ST_BUILDERS) {
        uint4 w[IF][2];
        int valid[IF]; const uint32_t *src[IF]; unsigned char *dst[IF];
        unsigned pend = 0;
#pragma unroll
        for (int v = 0; v < IF; ++v) {
            const int idx = idx0 + v * ST_BUILDERS;
            valid[v] = 0; src[v] = a.qx; dst[v] = C.bop;
            if (idx < C.nbch * 2 * NB) {
                const int b = idx % NB, g = idx / NB, slot = g >> 1, kh = g & 1;
                const int ent = C.ctab[6 + slot], kc = ent & 0xffff;
                valid[v] = min(8, max(0, (ent >> 16) - 8 * kh));
                src[v] = a.qx + (size_t)b * a.KOP + kc * 16 + kh * 8;
                dst[v] = C.bop + (size_t)slot * NB * 64 + (b >> 3) * 256 + kh * 128 + (b & 7) * 16;
                pend |= (valid[v] > 0 ? 1u : 0u) << v;
                valid[v] |= 16;                                         // in range: the item is written even when it is all padding
            }
            w[v][0] = w[v][1] = make_uint4(0u, 0u, 0u, 0u);
        }
        unsigned spins = 0;
        while (pend) {
#pragma unroll
            for (int v = 0; v < IF; ++v) if (pend >> v & 1) { w[v][0] = ld_relaxed4(src[v]); w[v][1] = ld_relaxed4(src[v] + 4); }
#pragma unroll
            for (int v = 0; v < IF; ++v)
                if (pend >> v & 1) {
                    const int nv = valid[v] & 15;
                    const uint32_t ww[8] = {w[v][0].x, w[v][0].y, w[v][0].z, w[v][0].w, w[v][1].x, w[v][1].y, w[v][1].z, w[v][1].w};
                    bool ok = true;
#pragma unroll
                    for (int e = 0; e < 8; ++e) ok = ok && (e >= nv || (ww[e] & 3u) == tag);
                    if (ok) pend &= ~(1u << v);
                }
            if (pend) {
                if ((++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                __nanosleep(ST_POLL_SLEEP);
            }
        }
#pragma unroll
        for (int v = 0; v < IF; ++v) {
            if (!(valid[v] & 16)) continue;
            const int nv = valid[v] & 15;
            const uint32_t ww[8] = {w[v][0].x, w[v][0].y, w[v][0].z, w[v][0].w, w[v][1].x, w[v][1].y, w[v][1].z, w[v][1].w};
            uint32_t hi[8], lo[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const float x = e < nv ? untag(ww[e]) : 0.f;
                hi[e] = bf16_rn_dev(x);
                lo[e] = bf16_rn_dev(x - __uint_as_float(hi[e] << 16));
            }
            *reinterpret_cast<uint4 *>(dst[v]) = make_uint4(hi[0] | (hi[1] << 16), hi[2] | (hi[3] << 16), hi[4] | (hi[5] << 16), hi[6] | (hi[7] << 16));
            *reinterpret_cast<uint4 *>(dst[v] + NB * 32) = make_uint4(lo[0] | (lo[1] << 16), lo[2] | (lo[3] << 16), lo[4] | (lo[5] << 16), lo[6] | (lo[7] << 16));
        }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_arrive(smem_u32(C.bars + SB_BRDY));
}

// ------------------------------------------------------------------------------------------------------------
// E: 128 threads = the 128 rows of a tile (thread <-> TMEM lane <-> row k of the CTA's block).
// ------------------------------------------------------------------------------------------------------------
template <int NB, bool TIMING>
__device__ __forceinline__ void stream_epilogue(const StreamArgs &a, const StreamCta &C, const int r, const int lane, const int w4)
{
    constexpr int U = NB >= 32 ? 32 : 16, NU = NB / U;
    const uint32_t lane_addr = C.tbase + ((uint32_t)(w4 * 32) << 16);
    const bool rowok = r < C.nb;
    const bool tmg = TIMING && r == 0;
    long long tm[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int n = 0; n < a.n_steps; ++n) {
        const uint32_t tag = ((uint32_t)n + 1u) & 3u;
        long long tk = tmg ? clock64() : 0;
        // ---- wait for q^n: warp 0 polls one word of every owner CTA this CTA reads from ---------------------
        if (w4 == 0) warp_poll_sentinels(C.ctab[6 + ST_BCH_MAX_DEV], lane, tag, C.s_abort, [&](int x) { return a.qx + C.ctab[7 + ST_BCH_MAX_DEV + x]; });
        if (w4 == 0) asm volatile("bar.arrive 4, 288;" ::: "memory");          // the owners build their share of the B operand
        bar_named(1, 128);
        if (tmg) { const long long t_ = clock64(); tm[7] += t_ - tk; }
        // ---- (a) the B operand of the step: this thread's share of the items (stream_build_B) ------------
        stream_build_B<NB, 4>(a, C, r, tag);
        if (tmg) { const long long t_ = clock64(); tm[0] += t_ - tk; tk = t_; }
        // ---- (b) q^n of the thread's own row, every sample -------------------------------------------------
        float qk[NB];
        {
            const uint32_t *src = a.qx + C.koff + r;
            uint32_t w[NB];
            unsigned long long pend = rowok ? (NB == 64 ? ~0ull : (1ull << NB) - 1ull) : 0ull;
            unsigned spins = 0;
            while (pend) {
#pragma unroll
                for (int b = 0; b < NB; ++b) if (pend >> b & 1ull) w[b] = ld_relaxed1(src + (size_t)b * a.KOP);
#pragma unroll
                for (int b = 0; b < NB; ++b) if ((pend >> b & 1ull) && (w[b] & 3u) == tag) pend &= ~(1ull << b);
                if (pend) {
                    if ((++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                    __nanosleep(ST_POLL_SLEEP);
                }
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) qk[b] = rowok ? untag(w[b]) : 0.f;
        }
        if (tmg) { const long long t_ = clock64(); tm[1] += t_ - tk; tk = t_; }
        // ---- (c) epilogue 1: partial G of every tile ---------------------------------------------------------
        for (int i = 0; i < C.ntiles; ++i) {
            const long long tw = tmg ? clock64() : 0;
            mbar_wait(smem_u32(C.bars + SB_ACCF + i), (unsigned)n & 1u, C.s_abort);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            if (tmg) tm[2] += clock64() - tw;
            uint32_t tu[NU][U];
            stream_load_t<NB, U, NU>(lane_addr, i, tu);
            float *ws = C.wsum + (size_t)(i & 1) * 4 * NB + w4 * NB;
#pragma unroll
            for (int u = 0; u < NU; ++u) {
                float p[U];
#pragma unroll
                for (int c = 0; c < U; ++c) p[c] = qk[u * U + c] * __uint_as_float(tu[u][c]);
                int col;
                const float s = warp_reduce_scatter<U>(p, lane, col);
                if (U == 32 || !(lane & 1)) ws[u * U + col] = s;
            }
            bar_named(1, 128);
            if (r < NB) {
                const float *w0 = C.wsum + (size_t)(i & 1) * 4 * NB + r;
                const float g = (w0[0] + w0[NB]) + (w0[2 * NB] + w0[3 * NB]);
                const int nm = C.ttab[i * a.tile_stride];
                st_relaxed1(a.Gx + ((size_t)nm * a.NKB + C.jb) * NB + r, tag_word(g, tag));
            }
        }
        if (tmg) { const long long t_ = clock64(); tm[3] += t_ - tk; tk = t_; }
        // ---- (d) epilogue 2: eta of the tile's mode, the row's partial force over the CTA's tiles -------------
        if (w4 == 0)
            warp_poll_sentinels(C.ntiles * a.NKB, lane, tag, C.s_abort, [&](int x) -> const uint32_t * {
                const int i = x / a.NKB, jb = x - i * a.NKB;
                const int *tt = C.ttab + i * a.tile_stride;
                return (tt[3] >> jb & 1) ? a.Gx + ((size_t)tt[0] * a.NKB + jb) * NB : nullptr;
            });
        bar_named(1, 128);
        if (tmg) { const long long t_ = clock64(); tm[4] += t_ - tk; }
        // eta[i][b] = s_n[b] * sum over the k blocks of the partial G, for every (tile, sample) of the CTA: the loads of a pair are in
        // flight together (one after the other they cost an L2 round trip each)
        for (int idx = r; idx < C.ntiles * NB; idx += 128) {
            const int i = idx / NB, b = idx - i * NB;
            const int *tt = C.ttab + i * a.tile_stride;
            const uint32_t *gp = a.Gx + (size_t)tt[0] * a.NKB * NB + b;
            uint32_t wv[ST_NKB_MAX_DEV];
            unsigned pend = (unsigned)tt[3], spins = 0;
            while (pend) {
#pragma unroll
                for (int jb = 0; jb < ST_NKB_MAX_DEV; ++jb) if (pend >> jb & 1) wv[jb] = ld_relaxed1(gp + (size_t)jb * NB);
#pragma unroll
                for (int jb = 0; jb < ST_NKB_MAX_DEV; ++jb) if ((pend >> jb & 1) && (wv[jb] & 3u) == tag) pend &= ~(1u << jb);
                if (pend) {
                    if ((++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                    __nanosleep(ST_POLL_SLEEP);
                }
            }
            float g = 0.f;
#pragma unroll
            for (int jb = 0; jb < ST_NKB_MAX_DEV; ++jb) if (tt[3] >> jb & 1) g += untag(wv[jb]);      // block order (deterministic)
            C.seta[idx] = C.ss[idx] * g;
        }
        bar_named(1, 128);
        float facc[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) facc[b] = 0.f;
        for (int i = 0; i < C.ntiles; ++i) {
            uint32_t tu[NU][U];
            stream_load_t<NB, U, NU>(lane_addr, i, tu);
            const float4 *ep = reinterpret_cast<const float4 *>(C.seta + i * NB);
#pragma unroll
            for (int u = 0; u < NU; ++u)
#pragma unroll
                for (int c4 = 0; c4 < U / 4; ++c4) {
                    const float4 e = ep[u * (U / 4) + c4];
                    const int b = u * U + 4 * c4;
                    facc[b] = fmaf(e.x, __uint_as_float(tu[u][4 * c4]), facc[b]);
                    facc[b + 1] = fmaf(e.y, __uint_as_float(tu[u][4 * c4 + 1]), facc[b + 1]);
                    facc[b + 2] = fmaf(e.z, __uint_as_float(tu[u][4 * c4 + 2]), facc[b + 2]);
                    facc[b + 3] = fmaf(e.w, __uint_as_float(tu[u][4 * c4 + 3]), facc[b + 3]);
                }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        mbar_arrive(smem_u32(C.bars + SB_ACCE));                         // the accumulators may be overwritten
        if (tmg) { const long long t_ = clock64(); tm[5] += t_ - tk; tk = t_; }
        // ---- (e) the row's partial force, every sample, to the owners of the row --------------------------------
        if (rowok) {
            uint32_t *dst = a.fx + ((size_t)C.c * 128 + r) * NB;
#pragma unroll
            for (int b = 0; b < NB; b += 4) st_tagged4(dst + b, facc[b], facc[b + 1], facc[b + 2], facc[b + 3], tag);
        }
        if (tmg) *reinterpret_cast<volatile long long *>(C.bars + 58) = clock64();
        mbar_arrive(smem_u32(C.bars + SB_FDONE));                        // the owners start polling for the step's forces only now
        if (tmg) { const long long t_ = clock64(); tm[6] += t_ - tk; }
    }
    if (tmg) for (int x = 0; x < 8; ++x) a.timing[(size_t)C.c * 16 + x] = tm[x];
}

// ------------------------------------------------------------------------------------------------------------
// O: 256 threads own rows [row0, row0 + rows) of the CTA's block, every sample.  Item = (row, 4 samples), LPQ lanes per item
// share the gather over the CTAs of the block; after the join lane `sub` updates EPL elements of the quad.
// ------------------------------------------------------------------------------------------------------------
template <int NB, int LPQ, bool TIMING, bool EXTRAS>
__device__ __forceinline__ void stream_owner_steps(const StreamArgs &a, const StreamCta &C, const int tl, const int n_begin, const int n_end, long long (&tm)[4], long long &tmx)
{
    constexpr int TL = 256, BQ = NB / 4, EPL = LPQ >= 4 ? 1 : 4 / LPQ;
    const int items = C.rows * BQ;
    const int NH = (C.nct + LPQ - 1) / LPQ;
    const bool tmg = TIMING && tl == 0;
    const double *cf = reinterpret_cast<const double *>(C.coef);
    const float *cw = reinterpret_cast<const float *>(cf + 3 * C.nel);
    for (int n = n_begin; n < n_end; ++n) {
        const uint32_t tag = ((uint32_t)n + 1u) & 3u, tag_next = ((uint32_t)n + 2u) & 3u;
        long long tk = tmg ? clock64() : 0;
        asm volatile("bar.sync 4, 288;" ::: "memory");                        // q^n complete (the epilogue warp that polls the sentinels arrives)
        stream_build_B<NB, (NB >= 64 ? 2 : 4)>(a, C, 128 + tl, tag);
        float2 *pk = C.pk + (size_t)(n & 1) * C.nel;
        // no force of step n is complete before the CTA's own epilogue has stored its part: sleep on a CTA barrier until then instead
        // of polling L2 through the whole MMA phase (148 x 192 lanes x 10 loads in flight would eat the bandwidth the H stream needs)
        mbar_wait(smem_u32(C.bars + SB_FDONE), (unsigned)n & 1u, C.s_abort);
        if (tmg) { const long long t_ = clock64(); tm[3] += t_ - tk; tk = t_; }
        if (tl < 32) warp_poll_sentinels(C.nct, tl, tag, C.s_abort, [&](int x) { return a.fx + ((size_t)(C.cta0 + x) * 128 + C.row0) * NB; });
        bar_named(2, TL);
        for (int base = 0; base < items * LPQ; base += TL) {
            const int idx = base + tl, item = idx / LPQ, sub = idx - item * LPQ;
            const bool act = item < items;
            const int rr = act ? item / BQ : 0, bq = act ? item - rr * BQ : 0;
            const int x0 = sub * NH, x1 = min(C.nct, x0 + NH);
            const uint32_t *fq = a.fx + ((size_t)C.cta0 * 128 + C.row0 + rr) * NB + 4 * bq;
            float4 fs = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int xx = x0; xx < x1; xx += MMA_GB) {                          // CTA order (deterministic)
                uint4 v[MMA_GB];
                const int cnt = min(MMA_GB, x1 - xx);
                unsigned pend = act ? (1u << cnt) - 1u : 0u, spins = 0;
                while (pend) {
#pragma unroll
                    for (int u = 0; u < MMA_GB; ++u)
                        if (pend >> u & 1) v[u] = ld_relaxed4(fq + (size_t)(xx + u) * 128 * NB);
#pragma unroll
                    for (int u = 0; u < MMA_GB; ++u)
                        if ((pend >> u & 1) && tags_ok(v[u], tag)) pend &= ~(1u << u);
                    if (pend) {
                        if ((++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                        __nanosleep(ST_POLL_SLEEP);
                    }
                }
                if (act) {
#pragma unroll
                    for (int u = 0; u < MMA_GB; ++u)
                        if (u < cnt) { fs.x += untag(v[u].x); fs.y += untag(v[u].y); fs.z += untag(v[u].z); fs.w += untag(v[u].w); }
                }
            }
            if (tmg && base == 0) { const long long t_ = clock64(); tm[0] += t_ - tk; tk = t_; tmx += t_ - *reinterpret_cast<volatile long long *>(C.bars + 58); }
#pragma unroll
            for (int m = 1; m < LPQ; m <<= 1) {
                fs.x += __shfl_xor_sync(FLOW_FULL, fs.x, m); fs.y += __shfl_xor_sync(FLOW_FULL, fs.y, m);
                fs.z += __shfl_xor_sync(FLOW_FULL, fs.z, m); fs.w += __shfl_xor_sync(FLOW_FULL, fs.w, m);
            }
            if (act && sub * EPL < 4) {
#pragma unroll
                for (int h = 0; h < EPL; ++h) {
                    const int hq = sub * EPL + h, be = 4 * bq + hq, e = rr * NB + be;
                    const double fd = (double)(hq == 0 ? fs.x : hq == 1 ? fs.y : hq == 2 ? fs.z : fs.w);
                    double qv = C.sq[e], vv = C.sv[e];
                    const double ckv = cf[e], ckq = cf[C.nel + e], cr = cf[2 * C.nel + e];
                    double fe = 0.0;
                    if (EXTRAS && be < a.batch) {
                        const int k = C.k0 + C.row0 + rr;
                        const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
                        if (a.traj) a.traj[((size_t)be * a.n_steps + n) * a.n_q + a.kperm[k]] = qv;
                        if (n == 0 && a.auto_start) vv = (cr != 0.0) ? a.astart[co] * qv + a.half_T2 * fd : 0.0;
                        if (a.fext) fe = (double)a.fext[(size_t)be * a.n_steps + n] * a.gain[(size_t)be * a.NQP + k];
                    }
                    vv = fma(ckv, vv, fma(-ckq, qv, cr * (fe - fd)));
                    qv += vv;
                    const float qn = (float)qv;
                    C.sq[e] = qv; C.sv[e] = vv;
                    st_relaxed1(a.qx + (size_t)be * a.KOP + C.koff + C.row0 + rr, tag_word(qn, tag_next));
                    pk[e] = make_float2(cw[e] * qn, qn * qn);
                }
            }
        }
        if (tmg) { const long long t_ = clock64(); tm[1] += t_ - tk; tk = t_; }
        bar_named(2, TL);
        if (tl < NB) {                                                          // pickup partial of q^{n+1}, sample tl, over the CTA's rows
            if (n >= 3 && tl < a.batch) {      // four buffers: the sample's pickup warp must have consumed q^{n-3} (it normally has, steps ago)
                unsigned spins = 0;
                while (ld_relaxed1(a.wflag + tl) < (unsigned)(n - 2)) {
                    if ((++spins & 255u) == 0 && (*C.s_abort || spins > (1u << 22))) { *C.s_abort = 1; break; }
                    __nanosleep(ST_POLL_SLEEP);
                }
            }
            float o = 0.f, nr = 0.f;
            for (int rr = 0; rr < C.rows; ++rr) { const float2 v = pk[rr * NB + tl]; o += v.x; nr += v.y; }
            unsigned long long *pp = a.px + (((size_t)((n + 1) & 3) * a.G + C.c) * NB + tl) * 2;
            const unsigned long long ep = (unsigned long long)((unsigned)n + 2u) << 32;
            const unsigned long long w0 = ep | __float_as_uint(o), w1 = ep | __float_as_uint(nr);
            asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(pp), "l"(w0), "l"(w1) : "memory");
        }
        if (tmg) { const long long t_ = clock64(); tm[2] += t_ - tk; }
    }
}

template <int NB, int LPQ, bool TIMING>
__device__ __forceinline__ void stream_owner(const StreamArgs &a, const StreamCta &C, const int tl)
{
    // ---- state, coefficients, q^0 and its pickup partials ----
    float2 *pk = C.pk + C.nel;                                                  // buffer 1: step 0 uses buffer 0
    double *cf = reinterpret_cast<double *>(C.coef);
    float *cw = reinterpret_cast<float *>(cf + 3 * C.nel);
    for (int e = tl; e < C.rows * NB; e += 256) {
        const int rr = e / NB, be = e - rr * NB, k = C.k0 + C.row0 + rr;
        double q = 0.0, v = 0.0, kvv = 0.0, kqq = 0.0, rc = 0.0; float wk = 0.f;
        if (be < a.batch) {
            q = a.q0[(size_t)be * a.NQP + k]; v = a.v0[(size_t)be * a.NQP + k];
            const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
            kvv = a.kv[co]; kqq = a.kq[co]; rc = a.r[co]; wk = a.w[co];
        }
        C.sq[e] = q; C.sv[e] = v; cf[e] = kvv; cf[C.nel + e] = kqq; cf[2 * C.nel + e] = rc; cw[e] = wk;
        const float qn = (float)q;
        st_relaxed1(a.qx + (size_t)be * a.KOP + C.koff + C.row0 + rr, tag_word(qn, 1u));
        pk[e] = make_float2(wk * qn, qn * qn);
    }
    bar_named(2, 256);
    if (tl < NB) {
        float o = 0.f, nr = 0.f;
        for (int rr = 0; rr < C.rows; ++rr) { const float2 v = pk[rr * NB + tl]; o += v.x; nr += v.y; }
        unsigned long long *pp = a.px + ((size_t)C.c * NB + tl) * 2;
        const unsigned long long w0 = (1ull << 32) | __float_as_uint(o), w1 = (1ull << 32) | __float_as_uint(nr);
        asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(pp), "l"(w0), "l"(w1) : "memory");
    }
    long long tm[4] = {0, 0, 0, 0}, tmx = 0;
    const bool extras = a.traj != nullptr || a.fext != nullptr;
    if (extras) stream_owner_steps<NB, LPQ, TIMING, true>(a, C, tl, 0, a.n_steps, tm, tmx);
    else {
        if (a.auto_start) stream_owner_steps<NB, LPQ, TIMING, true>(a, C, tl, 0, min(1, a.n_steps), tm, tmx);
        stream_owner_steps<NB, LPQ, TIMING, false>(a, C, tl, a.auto_start ? 1 : 0, a.n_steps, tm, tmx);
    }
    if (TIMING && tl == 0) { for (int x = 0; x < 4; ++x) a.timing[(size_t)C.c * 16 + 8 + x] = tm[x]; a.timing[(size_t)C.c * 16 + 14] = tmx; }
}

// W: CTA c writes out[b][n] for the samples b = c, c + G, ...: the sum over all CTAs of the pickup partials of q^n (a1 pickup + a6 write-out)
template <int NB>
__device__ __forceinline__ void stream_pickup_warp(const StreamArgs &a, const StreamCta &C, const int lane)
{
    constexpr int MAXS = 4;                                    // samples of one CTA: NB <= 64 samples over >= 16 CTAs; else the host refuses
    int sbad[MAXS];
#pragma unroll
    for (int x = 0; x < MAXS; ++x) sbad[x] = -1;
    for (int n = 0; n < a.n_steps; ++n) {
#pragma unroll
        for (int x = 0; x < MAXS; ++x) {
            const int b = C.c + x * a.G;
            if (b >= a.batch) break;
            float o = 0.f, nr = 0.f;
            for (int y = lane; y < a.G; y += 32) {
                const unsigned long long *pp = a.px + (((size_t)(n & 3) * a.G + y) * NB + b) * 2;
                unsigned long long w0, w1;
                unsigned spins = 0;
                do {
                    asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(w0), "=l"(w1) : "l"(pp) : "memory");
                    if ((unsigned)(w0 >> 32) == (unsigned)n + 1u && (unsigned)(w1 >> 32) == (unsigned)n + 1u) break;
                    if ((++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                    __nanosleep(ST_POLL_SLEEP);
                } while (true);
                o += __uint_as_float((unsigned)w0); nr += __uint_as_float((unsigned)w1);
            }
#pragma unroll
            for (int m = 16; m >= 1; m >>= 1) { o += __shfl_xor_sync(FLOW_FULL, o, m); nr += __shfl_xor_sync(FLOW_FULL, nr, m); }
            if (lane == 0) {
                a.out[(size_t)b * a.n_steps + n] = o;
                if (sbad[x] < 0 && !(isfinite(o) && isfinite(nr))) sbad[x] = n;
                st_relaxed1(a.wflag + b, (uint32_t)n + 1u);                    // q^n of sample b consumed: its buffer may be reused
            }
        }
        __syncwarp();
    }
    if (lane == 0) {
#pragma unroll
        for (int x = 0; x < MAXS; ++x) if (C.c + x * a.G < a.batch) a.first_bad[C.c + x * a.G] = sbad[x];
    }
}

template <int NB, bool TIMING>
__global__ void __launch_bounds__(ST_THREADS, 1) vk_stream_kernel(const StreamArgs a)
{
    extern __shared__ __align__(128) unsigned char st_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const StreamSmem L = stream_smem_layout(NB, a.rows_max, a.bch_max, a.tile_stride, a.NSTG, a.stage_bytes);
    StreamCta C;
    C.c = blockIdx.x;
    C.bars = reinterpret_cast<uint64_t *>(st_smem + L.bars);
    uint32_t *tptr = reinterpret_cast<uint32_t *>(C.bars + SB_TPTR);
    C.s_abort = reinterpret_cast<volatile int *>(C.bars + SB_ABORT);
    int *tab = reinterpret_cast<int *>(st_smem + L.tab);
    C.ctab = tab; C.ttab = tab + ST_CTA_STRIDE; C.blk = C.ttab + ST_TILES_MAX_DEV * a.tile_stride; C.bnct = C.blk + 4 * ST_NKB_MAX_DEV;
    C.ss = reinterpret_cast<float *>(st_smem + L.ss); C.wsum = reinterpret_cast<float *>(st_smem + L.wsum);
    C.seta = reinterpret_cast<float *>(st_smem + L.seta);
    C.sq = reinterpret_cast<double *>(st_smem + L.sq); C.sv = reinterpret_cast<double *>(st_smem + L.sv);
    C.coef = st_smem + L.coef; C.pk = reinterpret_cast<float2 *>(st_smem + L.pk);
    C.sbad = reinterpret_cast<int *>(st_smem + L.misc); C.wdone = reinterpret_cast<volatile int *>(st_smem + L.misc + 4);
    C.bop = st_smem + L.bop; C.ring = st_smem + L.ring;
    C.nel = (size_t)a.rows_max * NB;

    if (tid == 0) {
        for (int s = 0; s < a.NSTG; ++s) { mbar_init(smem_u32(C.bars + SB_FULL + s), 1); mbar_init(smem_u32(C.bars + SB_EMPTY + s), 1); }
        for (int s = 0; s < ST_TILES_MAX_DEV; ++s) mbar_init(smem_u32(C.bars + SB_ACCF + s), 1);
        mbar_init(smem_u32(C.bars + SB_ACCE), 128); mbar_init(smem_u32(C.bars + SB_BRDY), ST_BUILDERS); mbar_init(smem_u32(C.bars + SB_FDONE), 128);
        *C.s_abort = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < ST_CTA_STRIDE) tab[tid] = a.cta_tab[(size_t)C.c * ST_CTA_STRIDE + tid];
    if (tid < 4 * a.NKB) tab[ST_CTA_STRIDE + ST_TILES_MAX_DEV * a.tile_stride + tid] = a.blk[tid];
    if (tid < a.NKB) tab[ST_CTA_STRIDE + ST_TILES_MAX_DEV * a.tile_stride + 4 * ST_NKB_MAX_DEV + tid] = a.blk_nctas[tid];
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tptr)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    __syncthreads();
    C.tile0 = C.ctab[0]; C.ntiles = C.ctab[1]; C.jb = C.ctab[2]; C.nbch = C.ctab[3]; C.row0 = C.ctab[4]; C.rows = C.ctab[5];
    for (int x = tid; x < C.ntiles * a.tile_stride; x += blockDim.x) tab[ST_CTA_STRIDE + x] = a.tile_tab[(size_t)C.tile0 * a.tile_stride + x];
    C.k0 = C.blk[4 * C.jb]; C.nb = C.blk[4 * C.jb + 1]; C.koff = C.blk[4 * C.jb + 2]; C.cta0 = C.blk[4 * C.jb + 3]; C.nct = C.bnct[C.jb];
    C.x = C.c - C.cta0;
    for (int x = tid; x < C.ntiles * NB; x += blockDim.x) {                    // s_n[b] of the CTA's tiles
        const int i = x / NB, b = x - i * NB, nm = a.tile_tab[(size_t)(C.tile0 + i) * a.tile_stride];
        C.ss[x] = b < a.batch ? a.s[(size_t)(a.coeff_stride_phi ? b : 0) * a.n_phi + nm] : 0.f;
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    C.tbase = *tptr;

    if (warp >= 8) {
        if (NB >= 64) asm volatile("setmaxnreg.dec.sync.aligned.u32 120;"); else asm volatile("setmaxnreg.inc.sync.aligned.u32 152;");
        const int tl = tid - 256;
        if (a.LPQ == 1) stream_owner<NB, 1, TIMING>(a, C, tl);
        else if (a.LPQ == 2) stream_owner<NB, 2, TIMING>(a, C, tl);
        else if (a.LPQ == 4) stream_owner<NB, 4, TIMING>(a, C, tl);
        else stream_owner<NB, 8, TIMING>(a, C, tl);
    } else if (warp >= 4) {
        if (NB >= 64) asm volatile("setmaxnreg.inc.sync.aligned.u32 232;"); else asm volatile("setmaxnreg.inc.sync.aligned.u32 168;");
        stream_epilogue<NB, TIMING>(a, C, (warp & 3) * 32 + lane, lane, warp & 3);
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == 0) {
            // ---------------- P: the H stream of the CTA's tiles, every step, through the ring ----------------
            // ONE bulk copy per tile (its K chunks are contiguous in the stream: <= 56 KiB at C4): a cp.async.bulk costs ~670 cycles of the
            // SM's copy engine whatever its size (measured: 2 KiB and 32 KiB copies take the same time), so 8 or 16 KiB stages capped the
            // stream at 12-24 B/clk per SM and the step's MMAs waited for it (the whole MMA phase was this stream).
            if (lane == 0) {
                const uint32_t full0 = smem_u32(C.bars + SB_FULL), empty0 = smem_u32(C.bars + SB_EMPTY), ring0 = smem_u32(C.ring);
                const int NSTG = a.NSTG;
                int sg = 0; unsigned ph = 1;                                   // parity of the EMPTY phase to wait for
                for (int n = 0; n < a.n_steps; ++n)
                    for (int i = 0; i < C.ntiles; ++i) {
                        const int *tt = C.ttab + i * a.tile_stride;
                        const uint32_t bytes = (uint32_t)tt[1] * 8192u;
                        mbar_wait_fast(empty0 + 8 * sg, ph, C.s_abort);
                        mbar_expect_tx(full0 + 8 * sg, bytes);
                        tma_bulk_g2s(ring0 + sg * a.stage_bytes, a.A + (size_t)tt[2] * 4096, bytes, full0 + 8 * sg);
                        if (++sg == NSTG) { sg = 0; ph ^= 1u; }
                    }
            }
        } else if (warp == 1) {
            // ---------------- M: the MMAs ------------------------------------------------------------------------
            // ONE elected lane runs the whole role.  (A lane-0 branch makes ptxas wrap every tcgen05 instruction in an ELECT / R2UR /
            // branch loop; under elect.sync it knows a single thread is active.  An elect block per chunk or per tile costs ~130 and
            // ~300 cycles of issue latency each time it is entered -- measured beside ~45 cycles per MMA inside one.)
            if (elect_one_sync()) {
                const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(NB >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
                const uint32_t idesc2 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)((2 * NB) >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);   // N = 2 NB
                const uint32_t full0 = smem_u32(C.bars + SB_FULL), empty0 = smem_u32(C.bars + SB_EMPTY), accf0 = smem_u32(C.bars + SB_ACCF);
                const uint64_t dA0 = umma_desc(smem_u32(C.ring)), dB0 = umma_desc(smem_u32(C.bop));   // + (byte offset >> 4)
                const int NSTG = a.NSTG;
                int sg = 0; unsigned ph = 0;
                long long tmm = 0, tmw = 0;
                for (int n = 0; n < a.n_steps; ++n) {
                    mbar_wait(smem_u32(C.bars + SB_BRDY), (unsigned)n & 1u, C.s_abort);                    // q^n operand built
                    if (n > 0) mbar_wait(smem_u32(C.bars + SB_ACCE), (unsigned)(n - 1) & 1u, C.s_abort);    // last step's accumulators read
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const long long tk = TIMING ? clock64() : 0;
                    for (int i = 0; i < C.ntiles; ++i) {
                        const int *tt = C.ttab + i * a.tile_stride;
                        const int nch = tt[1];
                        const uint32_t td = C.tbase + (uint32_t)(i * StreamDual<NB>::TSTR);
                        {
                            const long long tw = TIMING ? clock64() : 0;
                            mbar_wait(full0 + 8 * sg, ph, C.s_abort);                          // the tile's chunks have landed
                            if (TIMING) tmw += clock64() - tw;
                        }
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        uint64_t dA = dA0 + (uint64_t)(sg * (a.stage_bytes >> 4));
                        for (int u = 0; u < nch; ++u, dA += 8192 / 16) {
                            const uint64_t dB = dB0 + (uint64_t)(tt[4 + u] * (NB * 64 / 16));
                            if (StreamDual<NB>::value) {
                                umma_bf16(td, dA, dB, idesc2, u > 0);                      // H_hi * [q_hi ; q_lo]  -> both column halves
                                umma_bf16(td, dA + 4096 / 16, dB, idesc, 1);               // H_lo * q_hi           -> first half
                            } else {
                                umma_bf16(td, dA, dB, idesc, u > 0);                       // hi * hi
                                umma_bf16(td, dA + 4096 / 16, dB, idesc, 1);               // lo * hi
                                umma_bf16(td, dA, dB + NB * 32 / 16, idesc, 1);            // hi * lo
                            }
                        }
                        umma_commit(empty0 + 8 * sg); umma_commit(accf0 + 8 * i);
                        if (++sg == NSTG) { sg = 0; ph ^= 1u; }
                    }
                    if (TIMING) tmm += clock64() - tk;
                }
                if (TIMING) { a.timing[(size_t)C.c * 16 + 12] = tmm; a.timing[(size_t)C.c * 16 + 13] = tmw; }
            }
            __syncwarp();
        } else if (warp == 2 && C.c < a.batch) {
            stream_pickup_warp<NB>(a, C, lane);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tid == 0 && *C.s_abort) *a.timeout_flag = 1;
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(C.tbase), "r"(512));
}

}  // namespace modal_dev
