// vk_mma.cuh -- batched MODAL_VK time loop on tcgen05 tensor cores, ONE persistent sm_100a kernel
// (layout in mma_schedule.hpp).
//
// Per time step, for up to 256 samples at once (two M tiles of 128):
//   t[b][(n,k)] = sum_r q[b][r] H^n[k][r]        tcgen05.mma kind::f16, bf16 hi/lo split, 3 MMAs per K chunk,
//                                                A = q chunk streamed by TMA from L2, B = H slab resident in
//                                                shared memory, D = t in TMEM (fp32), kept for both epilogues
//   G[b][n]  = sum_k q[b][k] t[b][(n,k)]         epilogue 1 (tcgen05.ld, one thread per sample), partial over
//                                                the CTA's RB rows k; summed over the k blocks through L2
//   eta      = s_n[b] G[b][n]                    (Eq. 9, C eliminated by PAPER.md:283)
//   f[b][k]  = sum_n eta[b][n] t[b][(n,k)]       epilogue 2, partial over the CTA's modes n; summed over
//                                                the n groups through L2 by the owner of (b, k)
//   fp64 delta-form update of the owner's (q, v) (Eq. 19-23), q republished as fp32 and
//   as bf16 hi/lo in operand layout; pickup out[b][n] = w . q^n.
// CTA (i,j) owns in-plane modes of group i and rows k of block j.
//
// Exchange between CTAs (no grid barrier, no atomics):
//  * partial G and partial f travel as TAGGED fp32 words: the two low mantissa bits carry (step+1) & 3, the
//    value is rounded to a multiple of 4 ulp (2^-22 relative, far below the 2^-17 of the split products).
//    A reader polls the data words themselves (ld.relaxed.gpu) until every tag matches: one L2 round trip,
//    no fence, no flag.  A word is only overwritten after q of the next step has been published by every
//    owner, i.e. after every reader of the previous value has consumed it, so a tag can never be mistaken
//    for the one written four steps earlier.
//  * the new state q feeds the TMA (async proxy), which cannot poll: owners store, one thread per
//    (CTA, tile) releases an epoch flag, the TMA warp of every CTA acquires the flags of all CTAs.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_flow.cuh"   // mbarrier / TMA / bounded-wait helpers

namespace modal_dev {

constexpr int MMA_NSTG = 6;          // q-operand ring stages (8 KiB each: 128 rows x 16 K x hi/lo) the layout fit assumes; the
constexpr int MMA_NSTG_MAX = 16;     // launch uses MmaArgs::NSTG stages (8 by default, <= 16) beside the compacted slab
// mbarrier indices: full[0..15] empty[16..31] acc_full[32,33] acc_empty[34,35] qready[36,37]; tmem pointer at word 40,
// abort word at 41, K-chunk list (64 ints) from word 44
constexpr int MB_FULL = 0, MB_EMPTY = 16, MB_ACCF = 32, MB_ACCE = 34, MB_QRDY = 36, MB_TPTR = 40, MB_ABORT = 41, MB_KLIST = 44;
constexpr int MMA_THREADS = 384;     // warpgroup 0: warps 0 / 2 TMA producers, warps 1 / 3 MMA issuers of tile 0 / 1 (56 registers
                                     // after setmaxnreg); warpgroups 1 / 2: epilogue + pickup of tile 0 / 1 (224 registers)
constexpr int MMA_FS = 8;            // words between the q flags of consecutive CTAs: one flag per 32-byte sector (C3 b256: 1 / 4 /
                                     // 8 / 16 / 32 words = 16.7 / 15.6 / 15.3 / 15.5 / 15.6 us per step; 147 stores to five lines serialise)
constexpr int MMA_FB = 11;           // 16-byte partial-force loads in flight per thread while polling (a thread keeps ~16 strong loads in flight)

struct MmaArgs {
    const uint16_t *slabs;      // [G][slab_bytes] bf16 hi/lo operand slabs of H: only the K chunks of klist, in list order
    int slab_bytes, NSTG;       // NSTG: ring stages of this launch (even, <= 16)
    int NKB, RB, NGRP, NG, NG4, NC, KC, KP, QS, G, nel_max;
    const int *nlist;           // [NGRP][NG] in-plane modes of each group (-1: empty)
    const int *klist, *kcnt;    // [G][KC], [G]: K chunks with a non-zero slab part (all others are skipped)
    int n_q, n_phi, NQP;
    int batch, n_steps, MT;     // batch <= 256; MT = M tiles in use
    int coeff_stride_q, coeff_stride_phi;
    const double *kv, *kq, *r, *astart;
    const float *s, *w;
    const double *q0, *v0;
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; const int *kperm; int *first_bad;
    // exchange (global, L2 resident)
    uint16_t *Qg;               // [2][KC][2][4096 B]   q as bf16 hi/lo operand chunks
    float *qf;                  // [256][QS]            q fp32
    uint32_t *Gx;               // [G][2][128][4*NG4]   partial G, tagged
    uint32_t *fx;               // [NGRP][2][128][QS]   partial f, tagged
    unsigned *qflag;            // [2][G][MMA_FS] epochs, one per (tile, CTA), each in its own 32-byte sector
    long long *timing;          // optional [G][8] cycle counters of tile 0 (MODAL_FLOW_TIMING)
};

__device__ __forceinline__ void set_flag(unsigned *p, unsigned epoch)
{
    asm volatile("fence.acq_rel.gpu;\n\tst.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(epoch) : "memory");
}
__device__ __forceinline__ void bar_named(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr)
{   // K-major, no swizzle: LBO = 128 B (K halves), SBO = 256 B (8-row groups), version 1
    return (uint64_t)((saddr >> 4) & 0x3fff) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld16_nowait(uint32_t taddr, uint32_t (&u)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]),
                   "=r"(u[8]), "=r"(u[9]), "=r"(u[10]), "=r"(u[11]), "=r"(u[12]), "=r"(u[13]), "=r"(u[14]), "=r"(u[15])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// The flags p[0 .. count): relaxed polls with a short sleep between rounds, then one ld.acquire.gpu per flag, which orders
// the q data behind the flags.  All CTAs poll the same few L2 lines while the owners try to store to them, so the
// polling rate matters (C3, us per step at batch 256 / 128): ld.acquire polls back to back 17.9 / 13.8 (each is followed
// by an L1 invalidate, which throttles them), relaxed polls back to back 21.3 / 13.3, relaxed + 400 ns sleep 16.6 / 12.8;
// a fence.acq_rel.gpu after relaxed polls measured slower (the MEMBAR stalls the epilogue warps of the other tile).
// (1.5 us sleep 16.3 / 12.6; sleeping through an estimate of the wait before the first poll 16.5 / 16.5: nanosleep overshoots)
constexpr unsigned MMA_POLL_SLEEP = 400;      // ns between polling rounds (with one flag per sector 0 / 200 / 400 / 800 ns: 15.5 / 15.4 / 15.3 / 15.5)
__device__ __forceinline__ void poll_flags(const unsigned *p, int lane, int count, unsigned epoch, volatile int *abortp)
{
    for (int base = lane; base < count; base += 256) {
        unsigned pend = 0, spins = 0;
#pragma unroll
        for (int u = 0; u < 8; ++u) if (base + 32 * u < count) pend |= 1u << u;
        while (pend) {
            unsigned v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (pend >> u & 1) asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v[u]) : "l"(p + (size_t)(base + 32 * u) * MMA_FS) : "memory");
#pragma unroll
            for (int u = 0; u < 8; ++u) if ((pend >> u & 1) && v[u] >= epoch) pend &= ~(1u << u);
            if (pend && (++spins & 1023u) == 0 && (*abortp || spins > (1u << 21))) { *abortp = 1; flow_timeout_flag = 1; break; }
            if (pend) __nanosleep(MMA_POLL_SLEEP);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (base + 32 * u < count) {
                // the value is not needed: the load is the acquire
                asm volatile("{\n\t.reg .b32 t;\n\tld.acquire.gpu.global.u32 t, [%0];\n\t}" ::"l"(p + (size_t)(base + 32 * u) * MMA_FS) : "memory");
            }
    }
}
__device__ __forceinline__ uint16_t bf16_rn_dev(float x)
{
    uint32_t u = __float_as_uint(x);
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}
// ---- tagged fp32 words -------------------------------------------------------------------------
__device__ __forceinline__ uint32_t tag_word(float x, uint32_t tag)
{
    uint32_t u = __float_as_uint(x);
    if ((u & 0x7f800000u) != 0x7f800000u) u += 2u;          // round to a multiple of 4 ulp; inf / nan stay non-finite
    return (u & ~3u) | tag;
}
__device__ __forceinline__ float untag(uint32_t w) { return __uint_as_float(w & ~3u); }
__device__ __forceinline__ void st_tagged4(uint32_t *p, float a, float b, float c, float d, uint32_t tag)
{
    asm volatile("st.relaxed.gpu.global.v4.b32 [%0], {%1,%2,%3,%4};"
                 ::"l"(p), "r"(tag_word(a, tag)), "r"(tag_word(b, tag)), "r"(tag_word(c, tag)), "r"(tag_word(d, tag)) : "memory");
}
__device__ __forceinline__ uint4 ld_relaxed4(const uint32_t *p)
{
    uint4 w;
    asm volatile("ld.relaxed.gpu.global.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "l"(p) : "memory");
    return w;
}
__device__ __forceinline__ uint32_t ld_relaxed1(const uint32_t *p)
{
    uint32_t w;
    asm volatile("ld.relaxed.gpu.global.b32 %0, [%1];" : "=r"(w) : "l"(p) : "memory");
    return w;
}
__device__ __forceinline__ bool tags_ok(const uint4 &w, uint32_t tag)
{
    return ((w.x & 3u) == tag) & ((w.y & 3u) == tag) & ((w.z & 3u) == tag) & ((w.w & 3u) == tag);
}

__host__ __device__ inline int mma_own_bytes(int nel_max) { return nel_max <= 512 ? 40 : 16; }
struct MmaSmem { size_t bars, own, sbad, cst, slab, ring, total; };
__host__ __device__ inline size_t mma_smem_fixed() { return 1024 + 256 * 4 + 256 * 64 + (size_t)MMA_NSTG * 8192 + 384; }
__host__ __device__ inline MmaSmem mma_smem_layout(int slab_bytes, int nel_max, int nstg)
{
    MmaSmem L; size_t o = 0;
    L.bars = o; o += 1024;                                 // mbarriers, tmem pointer, abort word, K-chunk list (MB_* above)
    L.own = o;  o += (size_t)2 * nel_max * mma_own_bytes(nel_max);   // owner state per tile: q, v (+ kv, kq, r if they fit), fp64 [nel_max] each
    L.sbad = o; o += 256 * 4;
    L.cst = o;  o += 256 * 64;                             // per epilogue thread: s_n[16] floats
    o = flow_align(o, 128);
    L.slab = o; o += (size_t)slab_bytes;
    o = flow_align(o, 128);
    L.ring = o; o += (size_t)nstg * 8192;
    L.total = o;
    return L;
}

// One epilogue group = 128 threads = one M tile of 128 samples (thread <-> TMEM lane <-> sample).
__device__ __forceinline__ void mma_epilogue_group(const MmaArgs &a, const int mt, const int c, const int i, const int j,
                                                   const int r, uint64_t *bars, double *own,
                                                   const uint32_t tbase, volatile int *s_abort, const int lane_base,
                                                   int *sbad, const int gw, const int lane, float *sreg)
{
    const int NC = a.NC, NG = a.NG, NG4 = a.NG4, QS = a.QS, NKB = a.NKB, NGRP = a.NGRP, B = a.batch, RB = a.RB, KC = a.KC;
    const int nch = (RB + 15) >> 4;
    const int b = mt * 128 + r;
    const bool valid = b < B;
    const float *sb = a.s + (size_t)(a.coeff_stride_phi ? (valid ? b : 0) : 0) * a.n_phi;
    // the (sample, k) elements this group owns for the update: rows r0..r1 of the tile, RB modes of block j
    const int r0 = 128 * i / NGRP, r1 = 128 * (i + 1) / NGRP, nel = (r1 - r0) * RB;
    double *sq = own, *sv = own + a.nel_max, *skv = own + 2 * a.nel_max, *skq = own + 3 * a.nel_max, *sr = own + 4 * a.nel_max;
    const bool csm = mma_own_bytes(a.nel_max) == 40;                                // update coefficients held in shared memory
    uint16_t *Qt = a.Qg + (size_t)mt * KC * 4096;                                  // chunk kc at + kc * 4096 (hi; lo at + 2048)
    // ---- owner state, coefficients, publish q^0 ----
    for (int e = r; e < nel; e += 128) {
        const int rr_ = e / RB, kk = e - rr_ * RB, re = r0 + rr_, be = mt * 128 + re, k = j * RB + kk;
        double q = 0.0, v = 0.0, kv = 0.0, kq = 0.0, rc = 0.0;
        if (be < B && k < a.n_q) {
            q = a.q0[(size_t)be * a.NQP + k]; v = a.v0[(size_t)be * a.NQP + k];
            const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
            kv = a.kv[co]; kq = a.kq[co]; rc = a.r[co];
            const float qfl = (float)q;
            a.qf[(size_t)be * QS + k] = qfl;
            const uint16_t hi = bf16_rn_dev(qfl), lo = bf16_rn_dev(qfl - __uint_as_float((uint32_t)hi << 16));
            const int k16 = k & 15;
            const int off = ((re >> 3) * 256 + (k16 >> 3) * 128 + (re & 7) * 16 + (k16 & 7) * 2) >> 1;
            uint16_t *Qc = Qt + (size_t)(k >> 4) * 4096;
            Qc[off] = hi; Qc[2048 + off] = lo;
        }
        sq[e] = q; sv[e] = v;
        if (csm) { skv[e] = kv; skq[e] = kq; sr[e] = rc; }
    }
    bar_named(2 + mt, 128);
    if (r == 0) set_flag(a.qflag + ((size_t)mt * a.G + c) * MMA_FS, 1u);
    for (int u = 0; u < 16; ++u) {                                                // [16][256]: conflict-free
        const int nn = u < NG ? a.nlist[i * NG + u] : -1;
        sreg[u * 256] = nn >= 0 ? sb[nn] : 0.f;
    }

    const uint32_t taddr0 = tbase + ((uint32_t)lane_base << 16) + (uint32_t)(mt * NC);
    const bool tmg = a.timing && r == 0 && mt == 0;
    long long *tm = a.timing + (size_t)c * 8;
    uint32_t *grow = a.Gx + ((size_t)(c * 2 + mt) * 128 + r) * (4 * NG4);
    const uint32_t *grd = a.Gx + ((size_t)((i * NKB) * 2 + mt) * 128 + r) * (4 * NG4);
    const size_t gstride = (size_t)2 * 128 * 4 * NG4;                               // words between consecutive k blocks
    uint32_t *frow = a.fx + ((size_t)(i * 2 + mt) * 128 + r) * QS + j * RB;
    const size_t fstride = (size_t)2 * 128 * QS;                                    // words between consecutive n groups
    const float *qrow = a.qf + (size_t)(valid ? b : 0) * QS + j * RB;

    for (int n = 0; n < a.n_steps; ++n) {
        const uint32_t tag = ((uint32_t)n + 1u) & 3u;
        long long tk = tmg ? clock64() : 0;
        mbar_wait(smem_u32(bars + MB_QRDY + mt), n & 1, s_abort);                  // q^n published by everybody
        if (tmg) { const long long t_ = clock64(); tm[0] += t_ - tk; tk = t_; }
        // ---- this sample's q over the rows of block j (operand of epilogue 1) ----
        float qb[32];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
            if (4 * u < RB) x = __ldcg(reinterpret_cast<const float4 *>(qrow) + u);
            qb[4 * u] = x.x; qb[4 * u + 1] = x.y; qb[4 * u + 2] = x.z; qb[4 * u + 3] = x.w;
        }
        // ---- a1 pickup + a6 write-out: out[b][n] = w . q^n for the samples b = c, c+G, ... of this tile ----
        for (int m = gw, b2 = c + gw * a.G; b2 < B; m += 4, b2 += 4 * a.G) {
            if (b2 / 128 != mt) continue;
            const float *wb = a.w + (size_t)(a.coeff_stride_q ? b2 : 0) * a.NQP;
            float o = 0.f, nrm = 0.f;
            for (int k = lane; k < a.n_q; k += 32) {
                const float qk = __ldcg(a.qf + (size_t)b2 * QS + k);
                o = fmaf(wb[k], qk, o); nrm = fmaf(qk, qk, nrm);
            }
#pragma unroll
            for (int sh = 16; sh >= 1; sh >>= 1) { o += __shfl_xor_sync(FLOW_FULL, o, sh); nrm += __shfl_xor_sync(FLOW_FULL, nrm, sh); }
            if (lane == 0) {
                a.out[(size_t)b2 * a.n_steps + n] = o;
                if (sbad[m] < 0 && !(isfinite(o) && isfinite(nrm))) sbad[m] = n;
            }
        }
        mbar_wait(smem_u32(bars + MB_ACCF + mt), n & 1, s_abort);                  // t of this tile is in TMEM
        if (tmg) { const long long t_ = clock64(); tm[1] += t_ - tk; tk = t_; }
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // ---- epilogue 1: partial G over the RB rows k of block j, four modes per pass ----
        for (int n4 = 0; n4 < NG4; ++n4) {
            float g4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int nl = 4 * n4 + u;
                if (nl < NG) {
                    uint32_t v0[16], v1[16];
                    tmem_ld16_nowait(taddr0 + nl * RB, v0);
                    if (nch > 1) tmem_ld16_nowait(taddr0 + nl * RB + 16, v1);
                    tmem_ld_wait();
#pragma unroll
                    for (int kk = 0; kk < 16; ++kk)
                        if (kk < RB) g4[u] = fmaf(qb[kk], __uint_as_float(v0[kk]), g4[u]);
                    if (nch > 1) {
#pragma unroll
                        for (int kk = 0; kk < 16; ++kk)
                            if (16 + kk < RB) g4[u] = fmaf(qb[16 + kk], __uint_as_float(v1[kk]), g4[u]);
                    }
                }
            }
            st_tagged4(grow + 4 * n4, g4[0], g4[1], g4[2], g4[3], tag);                   // G hop, send side
        }
        if (tmg) { const long long t_ = clock64(); tm[2] += t_ - tk; tk = t_; }
        float eta[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) eta[u] = 0.f;
        {
            // ---- G hop, receive side: gather the partial rows of all k blocks of this mode group ----
#pragma unroll
            for (int m = 0; m < 2; ++m)                                           // two float4 columns of the rows per batch
                if (2 * m < NG4)
                    for (int jj0 = 0; jj0 < NKB; jj0 += 8) {                        // k-block order (deterministic); 8 + 8 loads in flight
                        uint4 x[16];
                        const int cnt = min(8, NKB - jj0);
                        const unsigned lo8 = cnt >= 8 ? 0xffu : ((1u << cnt) - 1u);
                        unsigned pend = lo8 | (2 * m + 1 < NG4 ? lo8 << 8 : 0u), spins = 0;
                        while (pend) {
#pragma unroll
                            for (int u = 0; u < 16; ++u)
                                if (pend >> u & 1) x[u] = ld_relaxed4(grd + (size_t)(jj0 + (u & 7)) * gstride + 4 * (2 * m + (u >> 3)));
#pragma unroll
                            for (int u = 0; u < 16; ++u)
                                if ((pend >> u & 1) && tags_ok(x[u], tag)) pend &= ~(1u << u);
                            if (pend && (++spins & 1023u) == 0 && (*s_abort || spins > (1u << 21))) { *s_abort = 1; flow_timeout_flag = 1; break; }
                        }
#pragma unroll
                        for (int u = 0; u < 8; ++u)
                            if (u < cnt) {
                                eta[8 * m] += untag(x[u].x); eta[8 * m + 1] += untag(x[u].y);
                                eta[8 * m + 2] += untag(x[u].z); eta[8 * m + 3] += untag(x[u].w);
                                if (2 * m + 1 < NG4) {
                                    eta[8 * m + 4] += untag(x[u + 8].x); eta[8 * m + 5] += untag(x[u + 8].y);
                                    eta[8 * m + 6] += untag(x[u + 8].z); eta[8 * m + 7] += untag(x[u + 8].w);
                                }
                            }
                    }
        }
#pragma unroll
        for (int u = 0; u < 16; ++u) eta[u] *= sreg[u * 256];                             // eta_n = s_n G_n
        if (tmg) { const long long t_ = clock64(); tm[3] += t_ - tk; tk = t_; }
        // ---- epilogue 2: partial force over the modes n of group i, published as tagged words ----
        for (int ch = 0; ch < nch; ++ch) {
                float facc[16];
#pragma unroll
                for (int kk = 0; kk < 16; ++kk) facc[kk] = 0.f;
#pragma unroll
                for (int nl = 0; nl < 16; nl += 2)
                    if (nl < NG) {
                        uint32_t v0[16], v1[16];
                        tmem_ld16_nowait(taddr0 + nl * RB + ch * 16, v0);
                        if (nl + 1 < NG) tmem_ld16_nowait(taddr0 + (nl + 1) * RB + ch * 16, v1);
                        tmem_ld_wait();
#pragma unroll
                        for (int kk = 0; kk < 16; ++kk) {
                            facc[kk] = fmaf(eta[nl], __uint_as_float(v0[kk]), facc[kk]);
                            if (nl + 1 < NG) facc[kk] = fmaf(eta[nl + 1], __uint_as_float(v1[kk]), facc[kk]);
                        }
                    }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (ch * 16 + 4 * u < RB)
                        st_tagged4(frow + ch * 16 + 4 * u, facc[4 * u], facc[4 * u + 1], facc[4 * u + 2], facc[4 * u + 3], tag);
            }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        mbar_arrive(smem_u32(bars + MB_ACCE + mt));                                 // TMEM tile may be overwritten
        if (tmg) { const long long t_ = clock64(); tm[4] += t_ - tk; tk = t_; }
        // ---- f hop + owner update: group-ordered sum of the partial forces, a5 linear update (fp64, delta form) ----
        // A warp handles 16 quads (4 consecutive k of one owned row) per pass: lanes 0-15 gather the first half of the
        // groups, lanes 16-31 the second half, as 16-byte strong loads (few wide requests: a thread keeps only ~16 strong
        // loads in flight, so the 4-byte version needed three L2 round trips); the halves meet through one shuffle, then
        // every lane updates two elements of its quad.
        for (int qbase = 0; qbase < nel; qbase += 256) {
            const int hh = lane >> 4, e4 = qbase + 4 * (16 * gw + (lane & 15));
            const int rr_ = e4 / RB, kk = e4 - rr_ * RB, re = r0 + rr_, be = mt * 128 + re, kq0 = j * RB + kk;
            const bool qact = e4 < nel && be < B && kq0 < a.n_q;
            const int NH = (NGRP + 1) >> 1, g0 = hh * NH, g1 = min(NGRP, g0 + NH);
            const uint32_t *fq = a.fx + ((size_t)mt * 128 + (qact ? re : 0)) * QS + (qact ? kq0 : 0);
            float4 fs = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int ii0 = g0; ii0 < g1; ii0 += MMA_FB) {                           // group order (deterministic)
                uint4 x[MMA_FB];
                const int cnt = min(MMA_FB, g1 - ii0);
                unsigned pend = qact ? (1u << cnt) - 1u : 0u, spins = 0;
                {   // first round: every word, addresses by pointer increments
                    const uint32_t *p0 = fq + (size_t)ii0 * fstride;
#pragma unroll
                    for (int u = 0; u < MMA_FB; ++u)
                        if (u < cnt) { x[u] = ld_relaxed4(p0); p0 += fstride; }
#pragma unroll
                    for (int u = 0; u < MMA_FB; ++u)
                        if ((pend >> u & 1) && tags_ok(x[u], tag)) pend &= ~(1u << u);
                }
                while (pend) {                                                      // stragglers only
#pragma unroll
                    for (int u = 0; u < MMA_FB; ++u)
                        if (pend >> u & 1) x[u] = ld_relaxed4(fq + (size_t)(ii0 + u) * fstride);
#pragma unroll
                    for (int u = 0; u < MMA_FB; ++u)
                        if ((pend >> u & 1) && tags_ok(x[u], tag)) pend &= ~(1u << u);
                    if (pend && (++spins & 1023u) == 0 && (*s_abort || spins > (1u << 21))) { *s_abort = 1; flow_timeout_flag = 1; break; }
                }
#pragma unroll
                for (int u = 0; u < MMA_FB; ++u)
                    if (u < cnt) { fs.x += untag(x[u].x); fs.y += untag(x[u].y); fs.z += untag(x[u].z); fs.w += untag(x[u].w); }
            }
            __syncwarp();
            float4 fo;
            fo.x = __shfl_xor_sync(FLOW_FULL, fs.x, 16); fo.y = __shfl_xor_sync(FLOW_FULL, fs.y, 16);
            fo.z = __shfl_xor_sync(FLOW_FULL, fs.z, 16); fo.w = __shfl_xor_sync(FLOW_FULL, fs.w, 16);
            // first half + second half, in that order on both lanes; lane half hh updates elements 2hh, 2hh+1 of the quad
            const float f2[2] = {hh ? fo.z + fs.z : fs.x + fo.x, hh ? fo.w + fs.w : fs.y + fo.y};
            float qn[2] = {0.f, 0.f};                                               // the lane's two new values (0 beyond n_q: padding)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int e = e4 + 2 * hh + h, k = kq0 + 2 * hh + h;
                if (!(qact && k < a.n_q)) continue;
                const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
                const double fd = (double)f2[h], rr = csm ? sr[e] : a.r[co], kvv = csm ? skv[e] : a.kv[co], kqq = csm ? skq[e] : a.kq[co];
                double q = sq[e], v = sv[e];
                if (a.traj) a.traj[((size_t)be * a.n_steps + n) * a.n_q + a.kperm[k]] = q;
                if (n == 0 && a.auto_start)
                    v = (rr != 0.0) ? a.astart[co] * q + a.half_T2 * fd : 0.0;
                const double fe = a.fext ? (double)a.fext[(size_t)be * a.n_steps + n] * a.gain[(size_t)be * a.NQP + k] : 0.0;
                v = kvv * v - kqq * q + rr * (fe - fd);
                q += v;
                sq[e] = q; sv[e] = v;
                qn[h] = (float)q;
            }
            // publish the pair (k even, k + 1 < KP): one 8-byte fp32 store and one 4-byte store each for the bf16 hi and lo halves,
            // which are adjacent in the operand layout
            const int k0 = kq0 + 2 * hh;
            if (qact && k0 < a.n_q) {
                *reinterpret_cast<float2 *>(a.qf + (size_t)be * QS + k0) = make_float2(qn[0], qn[1]);
                const uint32_t h0 = bf16_rn_dev(qn[0]), h1 = bf16_rn_dev(qn[1]);
                const uint32_t l0 = bf16_rn_dev(qn[0] - __uint_as_float(h0 << 16)), l1 = bf16_rn_dev(qn[1] - __uint_as_float(h1 << 16));
                const int k16 = k0 & 15;
                const int off = (re >> 3) * 256 + (k16 >> 3) * 128 + (re & 7) * 16 + (k16 & 7) * 2;      // bytes, 4-aligned
                unsigned char *Qc = reinterpret_cast<unsigned char *>(Qt + (size_t)(k0 >> 4) * 4096);
                *reinterpret_cast<uint32_t *>(Qc + off) = h0 | (h1 << 16);
                *reinterpret_cast<uint32_t *>(Qc + 4096 + off) = l0 | (l1 << 16);
            }
        }
        if (tmg) { const long long t_ = clock64(); tm[5] += t_ - tk; tk = t_; }
        bar_named(2 + mt, 128);
        if (r == 0) set_flag(a.qflag + ((size_t)mt * a.G + c) * MMA_FS, (unsigned)n + 2u);
        if (tmg) { const long long t_ = clock64(); tm[6] += t_ - tk; tk = t_; }
    }
    if (lane == 0)
        for (int m = gw, b2 = c + gw * a.G; b2 < B; m += 4, b2 += 4 * a.G)
            if (b2 / 128 == mt) a.first_bad[b2] = sbad[m];
}

__global__ void __launch_bounds__(MMA_THREADS, 1) vk_mma_kernel(const MmaArgs a)
{
    extern __shared__ __align__(128) unsigned char mma_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x, i = c / a.NKB, j = c - i * a.NKB;
    const MmaSmem L = mma_smem_layout(a.slab_bytes, a.nel_max, a.NSTG);
    uint64_t *bars = reinterpret_cast<uint64_t *>(mma_smem + L.bars);      // indices MB_*
    uint32_t *tptr = reinterpret_cast<uint32_t *>(bars + MB_TPTR);
    volatile int *s_abort = reinterpret_cast<volatile int *>(bars + MB_ABORT);
    double *own = reinterpret_cast<double *>(mma_smem + L.own);
    int *sbad = reinterpret_cast<int *>(mma_smem + L.sbad);
    unsigned char *cst = mma_smem + L.cst;
    unsigned char *slab = mma_smem + L.slab, *ring = mma_smem + L.ring;

    if (tid == 0) {
        for (int s = 0; s < a.NSTG; ++s) { mbar_init(smem_u32(bars + MB_FULL + s), 1); mbar_init(smem_u32(bars + MB_EMPTY + s), 1); }
        for (int m = 0; m < 2; ++m) {
            mbar_init(smem_u32(bars + MB_ACCF + m), 1); mbar_init(smem_u32(bars + MB_ACCE + m), 128); mbar_init(smem_u32(bars + MB_QRDY + m), 1);
        }
        *s_abort = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int x = tid; x < 256; x += blockDim.x) sbad[x] = -1;
    if (tid < a.KC && tid < 64) reinterpret_cast<int *>(bars + MB_KLIST)[tid] = a.klist[(size_t)c * a.KC + tid];   // KC <= 64 (mma_layout)
    {   // H slab of this CTA: loaded once, resident for the whole run
        const uint4 *src = reinterpret_cast<const uint4 *>(a.slabs + (size_t)c * a.slab_bytes / 2);
        uint4 *dst = reinterpret_cast<uint4 *>(slab);
        for (int x = tid; x < a.slab_bytes / 16; x += blockDim.x) dst[x] = __ldg(src + x);
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tptr)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tbase = *tptr;
    const int MT = a.MT, KC = a.KC, NC = a.NC;

    const int KCA = a.kcnt[c];                     // K chunks with a non-zero slab part: the others are neither loaded nor multiplied
    const int *kl = reinterpret_cast<const int *>(bars + MB_KLIST);      // this CTA's chunk list, copied to shared memory above
    const int kc0 = c % KCA;                       // the chunks are walked from a per-CTA offset: spreads the q reads over the L2 slices
    if (warp >= 4) {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        const int mt = (warp - 4) >> 2, gw = warp & 3;
        if (mt < MT)
            mma_epilogue_group(a, mt, c, i, j, (warp & 3) * 32 + lane, bars, own + (size_t)mt * (mma_own_bytes(a.nel_max) / 8) * a.nel_max,
                               tbase, s_abort, (warp & 3) * 32, sbad, gw, lane, reinterpret_cast<float *>(cst) + (tid - 128));
    } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    // Warps 0 / 2 are the producers of tile 0 / 1, warps 1 / 3 the MMA issuers: the two tiles are independent pipelines
    // (own half of the ring stages when both tiles are in use), so a late q^n of one tile never holds up the other.
    const int mt = warp >> 1;
    const int NSH = MT > 1 ? a.NSTG / 2 : a.NSTG;
    if (mt < MT && (warp & 1) == 0) {
        // ---------------- producer: wait for q^n of the tile, stream it through the ring by TMA ----------
        int stage = 0; unsigned ph = 0;
        for (int n = 0; n < a.n_steps; ++n) {
            poll_flags(a.qflag + (size_t)mt * a.G * MMA_FS, lane, a.G, (unsigned)n + 1u, s_abort);
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(smem_u32(bars + MB_QRDY + mt));
                asm volatile("fence.proxy.async.global;" ::: "memory");
                for (int kx = 0; kx < KCA; ++kx) {
                    const int kc = kl[kx + kc0 < KCA ? kx + kc0 : kx + kc0 - KCA];
                    const int sg = NSH * mt + stage;
                    mbar_wait(smem_u32(bars + MB_EMPTY + sg), ph ^ 1, s_abort);
                    mbar_expect_tx(smem_u32(bars + MB_FULL + sg), 8192);
                    tma_bulk_g2s(smem_u32(ring + sg * 8192), a.Qg + ((size_t)mt * KC + kc) * 4096, 8192, smem_u32(bars + MB_FULL + sg));
                    if (++stage == NSH) { stage = 0; ph ^= 1; }
                }
            }
            __syncwarp();
        }
    } else if (mt < MT) {
        // ---------------- MMA issuer: one thread per tile ------------------------------------------------
        if (lane == 0) {
            const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(NC >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
            int stage = 0; unsigned ph = 0;
            const uint32_t td = tbase + (uint32_t)(mt * NC);
            for (int n = 0; n < a.n_steps; ++n) {
                mbar_wait(smem_u32(bars + MB_ACCE + mt), (n & 1) ^ 1, s_abort);         // epilogues of step n-1 left the tile
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                for (int kx = 0; kx < KCA; ++kx) {
                    const int kp = kx + kc0 < KCA ? kx + kc0 : kx + kc0 - KCA;          // position in the list = position in the slab
                    const int sg = NSH * mt + stage;
                    mbar_wait(smem_u32(bars + MB_FULL + sg), ph, s_abort);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t qa = smem_u32(ring + sg * 8192), hb = smem_u32(slab + (size_t)kp * 2 * NC * 32);
                    const uint64_t qhi = umma_desc(qa), qlo = umma_desc(qa + 4096);
                    const uint64_t hhi = umma_desc(hb), hlo = umma_desc(hb + NC * 32);
                    umma_bf16(td, qhi, hhi, idesc, kx > 0);
                    umma_bf16(td, qlo, hhi, idesc, 1);
                    umma_bf16(td, qhi, hlo, idesc, 1);
                    umma_commit(smem_u32(bars + MB_EMPTY + sg));                              // ring slot free when these MMAs retire
                    if (++stage == NSH) { stage = 0; ph ^= 1; }
                }
                umma_commit(smem_u32(bars + MB_ACCF + mt));                                // t of tile mt complete
            }
        }
    }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tbase), "r"(512));
}

}  // namespace modal_dev
