// vk_mma.cuh -- batched MODAL_VK time loop on tcgen05 tensor cores, ONE persistent sm_100a kernel for the whole
// batch (layout in mma_schedule.hpp).
//
// Per time step, for every M tile of 128 samples (any number of tiles in one launch):
//   t[b][(n,k)] = sum_r q[b][r] H^n[k][r]        tcgen05.mma kind::f16, bf16 hi/lo split, 3 MMAs per K chunk,
//                                                A = q chunk streamed by TMA from L2, B = H slab resident in
//                                                shared memory, D = t in a TMEM accumulator slot (fp32), kept
//                                                for both epilogues
//   G[b][n]  = sum_k q[b][k] t[b][(n,k)]         epilogue 1 (tcgen05.ld, one thread per sample), partial over
//                                                the rows k of the CTA's block; summed over the k blocks through L2
//   eta      = s_n[b] G[b][n]                    (Eq. 9, C eliminated by PAPER.md:283)
//   f[b][k]  = sum_n eta[b][n] t[b][(n,k)]       epilogue 2, partial over the CTA's modes n; summed over
//                                                the n groups through L2 by the owner of (b, k)
//   fp64 delta-form update of the owner's (q, v) (Eq. 19-23), q republished as fp32 and
//   as bf16 hi/lo in operand layout; pickup out[b][n] = w . q^n.
// CTA (i,j) owns the in-plane modes of group i and the rows k of block j.
//
// Roles (16 warps).  The stages of a tile-step are handled by DIFFERENT warps, each walking the tiles in the same
// order, so several tiles are in flight and a warp that waits on an exchange never holds up the tensor pipe:
//   warp 0      P  polls the q flags of the tile's source blocks, streams its K chunks through the ring by TMA
//   warp 1      M  one thread issues the MMAs of the tile into accumulator slot (tile mod S) and commits
//   warp 2      W  (block-0 CTAs) sums the pickup partials of its rows over the k blocks, writes the audio
//   warps 4-7   O  owners: gather the partial forces of the owned (row, k) elements, fp64 update, publish q
//   warps 8-15  E  two epilogue groups of 128 threads (thread <-> TMEM lane <-> sample), tiles alternate
//
// Exchange between CTAs (no grid barrier, no atomics; every wait is bounded):
//  * partial G and partial f travel as TAGGED fp32 words: the two low mantissa bits carry (step+1) & 3, the
//    value is rounded to a multiple of 4 ulp (2^-22 relative, far below the 2^-17 of the split products).
//    A reader polls the data words themselves (ld.relaxed.gpu) until every tag matches: one L2 round trip,
//    no fence, no flag.  Partial f of (tile, group, block) is rewritten only after q of the next step has been
//    flagged by EVERY owner of that block, i.e. after every reader consumed it.  Partial G is double-buffered by
//    step parity: a CTA can be at most one step ahead of a peer of its group (it needs the peer's next partial).
//  * the new state q feeds the TMA (async proxy), which cannot poll: owners store, one thread per
//    (CTA, tile) releases an epoch flag, warp P of every CTA that reads the block acquires its owners' flags.
//  * pickup partials (per row and k block) travel as {fp32, epoch} 64-bit words, double-buffered by step parity;
//    an owner releases its flag only after warp W of its CTA consumed the partials of the step before.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_flow.cuh"   // mbarrier / TMA / bounded-wait helpers

namespace modal_dev {

constexpr int MMA_THREADS = 512;
constexpr int MMA_NSTG_MAX = 16;     // q-operand ring stages (8 KiB each: 128 rows x 16 K x hi/lo)
constexpr int MMA_MT_MAX = 8;        // M tiles per launch (== modal_host::MMA_MT_MAX): wider batches run as consecutive launches
constexpr int MMA_FS = 8;            // words between consecutive q flags: one flag per 32-byte sector (profiles/r1_c3_b256.md)
constexpr int MMA_GB = 16;           // 16-byte strong loads a lane keeps in flight while gathering (all n groups of the C3 layout in one round trip)
constexpr int MMA_RB_MAX_DEV = 56;   // == modal_host::MMA_RB_MAX: rows k of a block (a sample's block of q lives in registers)
constexpr int MMA_NG_MAX_DEV = 8;    // == modal_host::MMA_NG_MAX: in-plane modes of a group
// mbarrier indices (64-bit words of the first shared-memory block)
constexpr int MB_FULL = 0, MB_EMPTY = 16, MB_ACCF = 32, MB_ACCE = 35, MB_QRDY = 38, MB_TPTR = 56, MB_ABORT = 57, MB_STAMP = 58, MB_RS = 60, MB_AG = 62;   // QRDY: one per tile (<= 16); RS / AG: cluster G exchange, one per slot
constexpr int MMA_TAB_OFF = 512;     // byte offset of the per-CTA tables inside the first block (ints): klist[64] nmode[8] fblk[16] blk[16][3]
constexpr int MMA_BARS_BYTES = 1536;

struct MmaArgs {
    const uint16_t *slabs;      // [G][slab_bytes] bf16 hi/lo operand slabs of H: only the K chunks of klist, in list order
    int slab_bytes, NSTG;
    int NKB, NGRP, NG, NG4, NC, S, RBT, RBQ, KC, KCL, G, rows_max, LPQ;
    int CL;                     // 1: the NKB CTAs of an n group form a thread-block cluster and exchange partial G through distributed shared memory
    const int *nlist;           // [NGRP][NG] in-plane modes of each group (-1: empty)
    const int *klist, *kcnt;    // [G][KCL], [G]
    const int *fblk, *fcnt;     // [G][16], [G]: blocks whose owners this CTA waits for (own block first)
    const int *blk;             // [NKB][3]: k0, nb, koff
    int n_q, n_phi, NQP;
    int batch, n_steps, MT;
    int coeff_stride_q, coeff_stride_phi;
    const double *kv, *kq, *r, *astart;
    const float *sT, *w;        // sT: s_n transposed [n_phi][sT_stride] (sample-major inside a mode: coalesced per warp)
    int sT_stride;
    const double *q0, *v0;
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; const int *kperm; int *first_bad;
    // exchange (global, L2 resident)
    uint16_t *Qop;              // [MT][KC][8192 B]                 q as bf16 operand chunks (hi 4 KiB, lo 4 KiB)
    float *qf;                  // [MT][NKB][RBQ][128][4]           q fp32, quads of 4 consecutive k of a block
    uint32_t *Gx;               // [2][MT][NGRP][NKB][128][4*NG4]   partial G, tagged, by step parity
    uint32_t *fx;               // [MT][NGRP][NKB][RBQ][128][4]     partial f, tagged
    unsigned *qflag;            // [MT][NKB][NGRP][MMA_FS]          epochs
    unsigned long long *px;     // [2][MT][NKB][128][2]             pickup partials {o, epoch}, {|q|^2, epoch}
    int *timeout_flag;          // per plan: set when a bounded wait gave up
    long long *timing;          // optional [G][16] cycle counters of tile 0
    long long *trace;           // optional [G][4][8] globaltimer stamps of tile 0 at steps 64..67 (phase boundaries; timing build)
};

struct MmaSmem { size_t bars, sq, sv, coef, pk, sbad, wdone, gex, slab, ring, total; };
__host__ __device__ inline MmaSmem mma_smem_layout(int slab_bytes, int MT, int rows_max, int RBQ, int nstg)
{
    MmaSmem L; size_t o = 0;
    const size_t nel = (size_t)rows_max * RBQ * 4;
    L.bars = o;  o += MMA_BARS_BYTES;
    L.sq = o;    o += (size_t)MT * nel * 8;
    L.sv = o;    o += (size_t)MT * nel * 8;
    L.coef = o;  o += (size_t)MT * nel * 28;                    // the owners' update coefficients, per tile: kv[nel], kq[nel], r[nel] fp64, w[nel] fp32
    L.pk = o;    o += (size_t)2 * 2 * rows_max * RBQ * 8;       // [team][buffer][row][quad] float2
    L.sbad = o;  o += (size_t)MT * rows_max * 4;
    L.wdone = o; o += (size_t)MMA_MT_MAX * 4;
    o = flow_align(o, 16);
    L.gex = o;   o += (size_t)2 * 2 * 128 * 32;                 // cluster G exchange: [reduce-scatter | all-gather][slot][128 x 8 floats]
    o = flow_align(o, 128);
    L.slab = o;  o += (size_t)slab_bytes;
    o = flow_align(o, 128);
    L.ring = o;  o += (size_t)nstg * 8192;
    L.total = o;
    return L;
}
__host__ __device__ inline size_t mma_smem_fixed() { return MMA_BARS_BYTES + 4096 + 1024; }   // besides slab, ring and owner state

__device__ __forceinline__ void set_flag(unsigned *p, unsigned epoch)
{
    // st.release = MEMBAR.ALL.GPU + strong store; fence.acq_rel + st.relaxed would add a CCTL.IVALL (L1 invalidate) the owner does not need
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(epoch) : "memory");
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
// ---- distributed shared memory (thread-block cluster) ---------------------------------------------
__device__ __forceinline__ uint32_t dsm_map(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// st.async: the store and the signal travel together -- the bytes are counted on the destination CTA's mbarrier (complete_tx), whose
// waiters see them when the phase completes; no fence, no separate arrive (a release-arrive per thread measured ~2 k cycles)
__device__ __forceinline__ void dsm_st_async4(uint32_t raddr, uint32_t rbar, float a, float b, float c, float d)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1,%2,%3,%4}, [%5];"
                 ::"r"(raddr), "r"(__float_as_uint(a)), "r"(__float_as_uint(b)), "r"(__float_as_uint(c)), "r"(__float_as_uint(d)), "r"(rbar) : "memory");
}
__device__ __forceinline__ void dsm_st_async1(uint32_t raddr, uint32_t rbar, float a)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(raddr), "r"(__float_as_uint(a)), "r"(rbar) : "memory");
}
__device__ __forceinline__ void dsm_wait(uint32_t bar, uint32_t parity, volatile int *abortp)
{
    uint32_t ok;
    unsigned spins = 0;
    const long long t0 = clock64();
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (!ok && (++spins & 63u) == 0 && (*abortp || clock64() - t0 > 3000000000LL)) { *abortp = 1; break; }
    } while (!ok);
}
__device__ __forceinline__ void mma_trace(const MmaArgs &a, int c, int n, int ev)
{
    if (a.trace && n >= 64 && n < 68) {
        long long g; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g));
        a.trace[((size_t)c * 4 + (n - 64)) * 8 + ev] = g;
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
__device__ __forceinline__ bool tags_ok(const uint4 &w, uint32_t tag)
{
    return ((w.x & 3u) == tag) & ((w.y & 3u) == tag) & ((w.z & 3u) == tag) & ((w.w & 3u) == tag);
}
__device__ __forceinline__ void mma_give_up(volatile int *s_abort, int *gflag) { *s_abort = 1; *gflag = 1; }

// The flags p[f * MMA_FS], f in the lane's share of [0, count): relaxed polls with a short sleep between rounds, then
// one ld.acquire.gpu per flag, which orders the q data behind the flags (profiles/r1_c3_b256.md: acquire polls
// are throttled by the L1 invalidate that follows each, back-to-back relaxed polls hammer the lines the owners store to).
constexpr unsigned MMA_POLL_SLEEP = 200;      // ns between polling rounds
__device__ __forceinline__ void poll_flag_list(const unsigned *base, const int *fblk, int fcnt, int NGRP, int lane,
                                               unsigned epoch, volatile int *s_abort)
{
    const int count = fcnt * NGRP;
    for (int f0 = 0; f0 < count; f0 += 128) {
        const unsigned *ptr[4];
        unsigned pend = 0, spins = 0;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int f = f0 + 32 * u + lane;
            ptr[u] = base;
            if (f < count) {
                const int bi = f / NGRP, i = f - bi * NGRP;
                ptr[u] = base + ((size_t)fblk[bi] * NGRP + i) * MMA_FS;
                pend |= 1u << u;
            }
        }
        const unsigned mine = pend;
        while (pend) {
            unsigned v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (pend >> u & 1) asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v[u]) : "l"(ptr[u]) : "memory");
#pragma unroll
            for (int u = 0; u < 4; ++u) if ((pend >> u & 1) && v[u] >= epoch) pend &= ~(1u << u);
            if (pend && (++spins & 255u) == 0 && (*s_abort || spins > (1u << 22))) { *s_abort = 1; break; }
            if (pend) __nanosleep(MMA_POLL_SLEEP);
        }
#ifndef MMA_NO_ACQUIRE
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (mine >> u & 1)      // the value is not needed: the load is the acquire
                asm volatile("{\n\t.reg .b32 t;\n\tld.acquire.gpu.global.u32 t, [%0];\n\t}" ::"l"(ptr[u]) : "memory");
#else
        (void)mine;
#endif
    }
}

// one try_wait on the fast path; the bounded loop only when the phase is not complete yet
__device__ __forceinline__ void mma_wait_fast(uint32_t bar, uint32_t parity, volatile int *abortp)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (!ok) mbar_wait(bar, parity, abortp);
}
__device__ __forceinline__ bool mma_elect_one()
{
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}

// CTA-uniform view of the kernel's shared memory and of the CTA's place in the grid
struct MmaCta {
    int c, i, j;                // CTA, n group, k block
    int k0, nb, koff, RBQj;     // this block: first internal mode, modes, operand offset, quads
    int NGa;                    // modes of this group
    int r0, rows;               // sample rows of a tile this CTA owns for the update
    int KCA;                    // K chunks this CTA multiplies
    uint64_t *bars;
    const int *kl, *nmode, *fb, *blk;     // tables in shared memory
    volatile int *s_abort;
    double *sq, *sv; unsigned char *coef; float2 *pk; int *sbad; volatile int *wdone;
    unsigned char *slab, *ring, *gex;
    uint32_t tbase;
    size_t nel;                 // owner-state elements per tile: rows_max * RBQ * 4
};

// ------------------------------------------------------------------------------------------------------------
// E: one epilogue group = 128 threads = the 128 samples of a tile (thread <-> TMEM lane <-> sample).
// The accumulator is read in units of 32 columns (one tcgen05.ld.32x32b.x32 each): unit u = (mode nl, 32-column part
// sp) with NSP parts per mode (NSP = 1: up to 8 modes of <= 32 rows; NSP = 2: up to 4 modes of <= 64 rows).  The
// load of unit u+1 is in flight while the FMAs of unit u run (double-buffered registers; tcgen05.wait::ld waits for
// every outstanding load of the thread, so the next load is issued right after the wait).
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t (&u)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]),
                   "=r"(u[8]), "=r"(u[9]), "=r"(u[10]), "=r"(u[11]), "=r"(u[12]), "=r"(u[13]), "=r"(u[14]), "=r"(u[15]),
                   "=r"(u[16]), "=r"(u[17]), "=r"(u[18]), "=r"(u[19]), "=r"(u[20]), "=r"(u[21]), "=r"(u[22]), "=r"(u[23]),
                   "=r"(u[24]), "=r"(u[25]), "=r"(u[26]), "=r"(u[27]), "=r"(u[28]), "=r"(u[29]), "=r"(u[30]), "=r"(u[31])
                 : "r"(taddr));
}

// E1: q of the own block, epilogue 1 (partial G), G hop send side -- every tile, in order.
template <int NSP, bool TIMING>
__device__ __forceinline__ void mma_epilogue_e1_tile(const MmaArgs &a, const MmaCta &C, const int r, const int lane_base, const int n, const int t,
                                                     const bool tmg, long long (&tm)[7])
{
    constexpr int NQ = 32 * NSP;                            // q values of the block a thread keeps (zero beyond the block)
    const int NG4 = a.NG4, NKB = a.NKB, NGRP = a.NGRP, RBT = a.RBT, RBQ = a.RBQ, S = a.S, MT = a.MT;
    const int nun = C.NGa * NSP;                            // units that hold data
    const size_t g_words = (size_t)128 * 4 * NG4;           // words of one (tile, group, block) partial-G array
    {
        const uint32_t tag = ((uint32_t)n + 1u) & 3u;
        {
            const int slot = t % S, uses = (MT - slot + S - 1) / S;
            const unsigned use = (unsigned)n * (unsigned)uses + (unsigned)(t / S);
            long long tk = tmg && t == 0 ? clock64() : 0;
            mbar_wait(smem_u32(C.bars + MB_QRDY + t), n & 1, C.s_abort);                 // q^n of the own block is published
            if (tmg && t == 0) { const long long t_ = clock64(); tm[0] += t_ - tk; tk = t_; mma_trace(a, C.c, n, 0); }
            // ---- this sample's q over the rows of block j (operand of epilogue 1), coalesced quads ----
            float q[NQ];
            {
                const float4 *qrow = reinterpret_cast<const float4 *>(a.qf) + ((size_t)(t * NKB + C.j) * RBQ) * 128 + r;
#pragma unroll
                for (int u = 0; u < NQ / 4; ++u) {
                    float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (u < C.RBQj) x = __ldcg(qrow + (size_t)u * 128);
                    q[4 * u] = x.x; q[4 * u + 1] = x.y; q[4 * u + 2] = x.z; q[4 * u + 3] = x.w;
                }
            }
            mbar_wait(smem_u32(C.bars + MB_ACCF + slot), use & 1u, C.s_abort);            // t of this tile is in TMEM
            if (tmg && t == 0) { const long long t_ = clock64(); tm[1] += t_ - tk; tk = t_; mma_trace(a, C.c, n, 1); }
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t taddr0 = C.tbase + ((uint32_t)lane_base << 16) + (uint32_t)(slot * a.NC);
            // ---- epilogue 1: partial G over the rows k of block j ----
            float g[MMA_NG_MAX_DEV];
#pragma unroll
            for (int nl = 0; nl < MMA_NG_MAX_DEV; ++nl) g[nl] = 0.f;
            {   // straight-line double buffering: every iteration handles units u, u + 1 and always issues the next loads
                // (addresses clamped to the last unit, whose reload is harmless), so no load sits under a branch
                uint32_t v0[32], v1[32];
                const int ulast = nun - 1;
                tmem_ld32_nowait(taddr0, v0);
                if (tmg && t == 0) { tmem_ld_wait(); tm[5] += clock64() - tk; }
                for (int u = 0; u < nun; u += 2) {
                    const int u1 = min(u + 1, ulast), u2 = min(u + 2, ulast);
                    tmem_ld_wait();
                    tmem_ld32_nowait(taddr0 + (u1 / NSP) * RBT + (u1 % NSP) * 32, v1);
                    float p0[4] = {0.f, 0.f, 0.f, 0.f}, p1[4] = {0.f, 0.f, 0.f, 0.f};      // four chains each: the FMA latency is not on the path
#pragma unroll
                    for (int kk = 0; kk < 32; ++kk) p0[kk & 3] = fmaf(q[kk], __uint_as_float(v0[kk]), p0[kk & 3]);
                    tmem_ld_wait();
                    tmem_ld32_nowait(taddr0 + (u2 / NSP) * RBT + (u2 % NSP) * 32, v0);
#pragma unroll
                    for (int kk = 0; kk < 32; ++kk) p1[kk & 3] = fmaf(q[(NSP - 1) * 32 + kk], __uint_as_float(v1[kk]), p1[kk & 3]);
                    const float acc0 = (p0[0] + p0[1]) + (p0[2] + p0[3]);
                    float acc1 = (p1[0] + p1[1]) + (p1[2] + p1[3]);
                    if (u + 1 > ulast) acc1 = 0.f;
                    const int m0 = u / NSP, m1 = (u + 1) / NSP;              // NSP = 2: both units belong to mode u / 2
#pragma unroll
                    for (int m = 0; m < MMA_NG_MAX_DEV; ++m) g[m] += (m == m0 ? acc0 : 0.f) + (m == m1 ? acc1 : 0.f);
                }
                tmem_ld_wait();
            }
            if (tmg && t == 0) tm[6] += clock64() - tk;
            // ---- G hop, send side ----
            if (a.CL) {
                // cluster of the group's k blocks: row r is summed by CTA r / RPR (reduce-scatter over the rows); the partials go
                // straight into that CTA's shared memory, the arrival on its mbarrier releases them (no polling, no L2)
                const int RPR = 128 / NKB, jr = r / RPR, lr = r - jr * RPR;
                const uint32_t dst = dsm_map(smem_u32(C.gex) + (uint32_t)(((slot * NKB + C.j) * RPR + lr) * 32), (uint32_t)jr);
                const uint32_t rbar = dsm_map(smem_u32(C.bars + MB_RS + slot), (uint32_t)jr);
                dsm_st_async4(dst, rbar, g[0], g[1], g[2], g[3]);
                if (NG4 > 1) dsm_st_async4(dst + 16, rbar, g[4], g[5], g[6], g[7]);
            } else {
                // through L2 (buffer of this step's parity): tagged words the peers poll
                uint32_t *gx = a.Gx + ((size_t)(n & 1) * MT + t) * NGRP * NKB * g_words;
                uint32_t *grow = gx + ((size_t)C.i * NKB + C.j) * g_words + (size_t)r * 4 * NG4;
                st_tagged4(grow, g[0], g[1], g[2], g[3], tag);
                if (NG4 > 1) st_tagged4(grow + 4, g[4], g[5], g[6], g[7], tag);
            }
            if (tmg && t == 0) { const long long t_ = clock64(); tm[2] += t_ - tk; tk = t_; mma_trace(a, C.c, n, 2); }
        }
    }
}

// E2: G hop receive side, eta, epilogue 2 (partial force), release of the accumulator slot -- every tile, in order.
// Runs on its own warpgroup, so the wait for the peers' partial G never holds up epilogue 1 of the next tile.
template <int NSP, bool TIMING>
__device__ __forceinline__ void mma_epilogue_e2_tile(const MmaArgs &a, const MmaCta &C, const int r, const int lane_base, const int n, const int t,
                                                     const bool tmg, long long (&tm)[7], const int wg)
{
    const int NG4 = a.NG4, NKB = a.NKB, NGRP = a.NGRP, B = a.batch, RBT = a.RBT, RBQ = a.RBQ, S = a.S, MT = a.MT;
    const size_t g_words = (size_t)128 * 4 * NG4;
    {
        const uint32_t tag = ((uint32_t)n + 1u) & 3u;
        {
            const int slot = t % S, uses = (MT - slot + S - 1) / S;
            const unsigned use = (unsigned)n * (unsigned)uses + (unsigned)(t / S);
            const int b = t * 128 + r;
            const bool valid = b < B;
            const uint32_t taddr0 = C.tbase + ((uint32_t)lane_base << 16) + (uint32_t)(slot * a.NC);
            const uint32_t *gx = a.Gx + ((size_t)(n & 1) * MT + t) * NGRP * NKB * g_words;
            mbar_wait(smem_u32(C.bars + MB_ACCF + slot), use & 1u, C.s_abort);            // t of this tile is in TMEM
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            float sc[MMA_NG_MAX_DEV];                                                      // s_n of this sample: in flight during the hop
#pragma unroll
            for (int u = 0; u < MMA_NG_MAX_DEV; ++u) {
                const int nn = u < a.NG ? C.nmode[u] : -1;
                sc[u] = nn >= 0 ? __ldg(a.sT + (size_t)nn * a.sT_stride + (a.coeff_stride_phi && valid ? b : 0)) : 0.f;
            }
            long long tk = tmg && t == 0 ? clock64() : 0;
            // ---- G hop, receive side: G_n of this sample summed over the k blocks of the group, block order ----
            float eta[MMA_NG_MAX_DEV];
#pragma unroll
            for (int u = 0; u < MMA_NG_MAX_DEV; ++u) eta[u] = 0.f;
            if (a.CL) {
                // reduce: this CTA sums RPR rows x 8 modes over the NKB sources, broadcasts the totals into every peer's shared memory
                const int RPR = 128 / NKB;
                const uint32_t gex = smem_u32(C.gex);
                if (r == 0) {      // arm this tile-step's phases: the bytes the peers send (they may already have arrived: the count is signed)
                    mbar_expect_tx(smem_u32(C.bars + MB_RS + slot), 128u * 16u * (uint32_t)NG4);
                    mbar_expect_tx(smem_u32(C.bars + MB_AG + slot), 4096u);
                }
                dsm_wait(smem_u32(C.bars + MB_RS + slot), use & 1u, C.s_abort);
                const float *rs = reinterpret_cast<const float *>(C.gex) + (size_t)slot * 1024;
                for (int item = r; item < RPR * 8; item += 128) {
                    float tot = 0.f;
                    for (int src = 0; src < NKB; ++src) tot += rs[src * RPR * 8 + item];                 // item = local row * 8 + mode
                    const uint32_t off = (uint32_t)(8192 + slot * 4096 + (C.j * RPR * 8 + item) * 4);  // all-gather area: [slot][row][mode]
                    for (int peer = 0; peer < NKB; ++peer)
                        dsm_st_async1(dsm_map(gex + off, (uint32_t)peer), dsm_map(smem_u32(C.bars + MB_AG + slot), (uint32_t)peer), tot);
                }
                dsm_wait(smem_u32(C.bars + MB_AG + slot), use & 1u, C.s_abort);
                const float4 *ag = reinterpret_cast<const float4 *>(C.gex + 8192 + slot * 4096 + r * 32);
                const float4 x0 = ag[0], x1 = ag[1];
                eta[0] = x0.x; eta[1] = x0.y; eta[2] = x0.z; eta[3] = x0.w; eta[4] = x1.x; eta[5] = x1.y; eta[6] = x1.z; eta[7] = x1.w;
            } else
            {
                const uint32_t *grd = gx + (size_t)C.i * NKB * g_words + (size_t)r * 4 * NG4;
                for (int jj0 = 0; jj0 < NKB; jj0 += 8) {
                    uint4 x[16];
                    const int cnt = min(8, NKB - jj0);
                    unsigned pend = 0, spins = 0;
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (u < cnt) pend |= (1u << u) | (NG4 > 1 ? 1u << (u + 8) : 0u);
                    while (pend) {
#pragma unroll
                        for (int u = 0; u < 16; ++u)
                            if (pend >> u & 1) x[u] = ld_relaxed4(grd + (size_t)(jj0 + (u & 7)) * g_words + 4 * (u >> 3));
#pragma unroll
                        for (int u = 0; u < 16; ++u)
                            if ((pend >> u & 1) && tags_ok(x[u], tag)) pend &= ~(1u << u);
                        if (pend && (++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (u < cnt) {
                            {
                                eta[0] += untag(x[u].x); eta[1] += untag(x[u].y); eta[2] += untag(x[u].z); eta[3] += untag(x[u].w);
                                if (NG4 > 1) {
                                    eta[4] += untag(x[u + 8].x); eta[5] += untag(x[u + 8].y);
                                    eta[6] += untag(x[u + 8].z); eta[7] += untag(x[u + 8].w);
                                }
                            }
                        }
                }
            }
#pragma unroll
            for (int u = 0; u < MMA_NG_MAX_DEV; ++u) eta[u] *= sc[u];                       // eta_n = s_n G_n
            if (tmg && t == 0) { const long long t_ = clock64(); tm[3] += t_ - tk; tk = t_; mma_trace(a, C.c, n, 3); }
            // ---- epilogue 2: partial force over the modes n of group i, published as tagged quads ----
            uint32_t *frow = a.fx + ((((size_t)t * NGRP + C.i) * NKB + C.j) * RBQ) * 512 + (size_t)r * 4;
#pragma unroll
            for (int sp = 0; sp < NSP; ++sp) {
                float facc[32];
#pragma unroll
                for (int kk = 0; kk < 32; ++kk) facc[kk] = 0.f;
                uint32_t v0[32], v1[32];
                const int nlast = C.NGa - 1;
                tmem_ld32_nowait(taddr0 + sp * 32, v0);
                for (int nl = 0; nl < C.NGa; nl += 2) {
                    const int n1 = min(nl + 1, nlast), n2 = min(nl + 2, nlast);
                    float e0 = 0.f, e1 = 0.f;
#pragma unroll
                    for (int m = 0; m < MMA_NG_MAX_DEV; ++m) { e0 = m == nl ? eta[m] : e0; e1 = m == nl + 1 ? eta[m] : e1; }
                    if (nl + 1 > nlast) e1 = 0.f;
                    tmem_ld_wait();
                    tmem_ld32_nowait(taddr0 + n1 * RBT + sp * 32, v1);
#pragma unroll
                    for (int kk = 0; kk < 32; ++kk) facc[kk] = fmaf(e0, __uint_as_float(v0[kk]), facc[kk]);
                    tmem_ld_wait();
                    tmem_ld32_nowait(taddr0 + n2 * RBT + sp * 32, v0);
#pragma unroll
                    for (int kk = 0; kk < 32; ++kk) facc[kk] = fmaf(e1, __uint_as_float(v1[kk]), facc[kk]);
                }
                tmem_ld_wait();
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    if (8 * sp + u < C.RBQj)
                        st_tagged4(frow + (size_t)(8 * sp + u) * 512, facc[4 * u], facc[4 * u + 1], facc[4 * u + 2], facc[4 * u + 3], tag);
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            mbar_arrive(smem_u32(C.bars + MB_ACCE + slot));                              // the accumulator slot may be overwritten
            if (tmg && t == 0) { const long long t_ = clock64(); tm[4] += t_ - tk; tk = t_; *reinterpret_cast<volatile long long *>(C.bars + MB_STAMP) = t_; mma_trace(a, C.c, n, 4); }
        }
    }
}

// The two epilogue warpgroups.  Up to two tiles: warpgroup 0 runs phase 1 (q, epilogue 1, G send) and warpgroup 1 phase 2 (G
// receive, epilogue 2) of every tile, so a tile's two TMEM passes overlap the other tile's.  More tiles: warpgroup w runs both phases
// of the tiles t = w, w + 2, ... (measured on C3, us per step at batch 128 / 256 / 1024: split 11.7 / 13.5 / 41.5, per-tile 12.2 / 14.3 / 34.4).
template <int NSP, bool TIMING>
__device__ __forceinline__ void mma_epilogue_warpgroup(const MmaArgs &a, const MmaCta &C, const int w, const int r, const int lane_base)
{
    const bool tmg = TIMING && r == 0;
    long long tm[7] = {0, 0, 0, 0, 0, 0, 0};               // phase cycles of tile 0, kept in registers (a global update per phase would add an L2 round trip to it)
    if (a.MT <= 2) {
        for (int n = 0; n < a.n_steps; ++n)
            for (int t = 0; t < a.MT; ++t) {
                if (w == 0) mma_epilogue_e1_tile<NSP, TIMING>(a, C, r, lane_base, n, t, tmg, tm);
                else mma_epilogue_e2_tile<NSP, TIMING>(a, C, r, lane_base, n, t, tmg, tm, w);
            }
    } else {
        for (int n = 0; n < a.n_steps; ++n)
            for (int t = w; t < a.MT; t += 2) {
                mma_epilogue_e1_tile<NSP, TIMING>(a, C, r, lane_base, n, t, tmg && w == 0, tm);
                mma_epilogue_e2_tile<NSP, TIMING>(a, C, r, lane_base, n, t, tmg && w == 0, tm, w);
            }
    }
    if (tmg && (a.MT <= 2 || w == 0)) {
        if (a.MT > 2 || w == 0) { for (int x = 0; x < 3; ++x) a.timing[(size_t)C.c * 16 + x] = tm[x]; a.timing[(size_t)C.c * 16 + 5] = tm[5]; a.timing[(size_t)C.c * 16 + 6] = tm[6]; }
        if (a.MT > 2 || w == 1) { a.timing[(size_t)C.c * 16 + 3] = tm[3]; a.timing[(size_t)C.c * 16 + 4] = tm[4]; }
    }
}


// ------------------------------------------------------------------------------------------------------------
// O: owners.  A team of TS warps handles the tiles t = team, team + NTEAM, ...: for every owned (row, quad of 4 k)
// gathers the partial forces of all n groups (16-byte strong loads, all in flight, group order), applies the a5
// linear update in fp64 delta form and republishes q.  LPQ lanes share a quad (each gathers a part of the groups).
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mma_publish(const MmaArgs &a, const MmaCta &C, int t, int re, int qd, int h0, int cnt, const float *qn)
{
    // qn[0..cnt): new values of elements 4*qd + h0 .. of row re in block j (cnt = 4, 2 or 1; h0 multiple of cnt)
    float *qf = a.qf + ((((size_t)t * a.NKB + C.j) * a.RBQ + qd) * 128 + re) * 4 + h0;
    const int kop = C.koff + 4 * qd + h0, k16 = kop & 15;
    unsigned char *Qc = reinterpret_cast<unsigned char *>(a.Qop) + ((size_t)t * a.KC + (kop >> 4)) * 8192 +
                        (re >> 3) * 256 + (k16 >> 3) * 128 + (re & 7) * 16 + (k16 & 7) * 2;
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const float x = u < cnt ? qn[u] : 0.f;
        hi[u] = bf16_rn_dev(x);
        lo[u] = bf16_rn_dev(x - __uint_as_float(hi[u] << 16));
    }
    if (cnt == 4) {
        *reinterpret_cast<float4 *>(qf) = make_float4(qn[0], qn[1], qn[2], qn[3]);
        *reinterpret_cast<uint2 *>(Qc) = make_uint2(hi[0] | (hi[1] << 16), hi[2] | (hi[3] << 16));
        *reinterpret_cast<uint2 *>(Qc + 4096) = make_uint2(lo[0] | (lo[1] << 16), lo[2] | (lo[3] << 16));
    } else if (cnt == 2) {
        *reinterpret_cast<float2 *>(qf) = make_float2(qn[0], qn[1]);
        *reinterpret_cast<uint32_t *>(Qc) = hi[0] | (hi[1] << 16);
        *reinterpret_cast<uint32_t *>(Qc + 4096) = lo[0] | (lo[1] << 16);
    } else {
        *qf = qn[0];
        *reinterpret_cast<uint16_t *>(Qc) = (uint16_t)hi[0];
        *reinterpret_cast<uint16_t *>(Qc + 4096) = (uint16_t)lo[0];
    }
}

// Steps [n_begin, n_end) of an owner team.  EXTRAS: trajectory output, external force or the second-order start at n = 0 are
// in use (a separate instance keeps their registers out of the common path).
template <int LPQ, bool TIMING, bool EXTRAS>
__device__ __forceinline__ void mma_owner_steps(const MmaArgs &a, const MmaCta &C, const int team, const int NTEAM, const int tl, const int TL,
                                                const int n_begin, const int n_end, unsigned &it, long long (&tm)[4], long long &tmx)
{
    const int NGRP = a.NGRP, NKB = a.NKB, RBQ = a.RBQ, B = a.batch, MT = a.MT;
    const int items = C.rows * C.RBQj;
    constexpr int EPL = 4 / LPQ;
    const int NH = (NGRP + LPQ - 1) / LPQ;
    const size_t fstride = (size_t)NKB * RBQ * 512;
    const bool tmg = TIMING && team == 0 && tl == 0;
    for (int n = n_begin; n < n_end; ++n) {
        const uint32_t tag = ((uint32_t)n + 1u) & 3u;
        for (int t = team; t < MT; t += NTEAM, ++it) {
            double *sq = C.sq + (size_t)t * C.nel, *sv = C.sv + (size_t)t * C.nel;
            // the row leaders read pk after the team barrier of this tile-step; the buffer is written again two
            // tile-steps later, i.e. after the barrier of the next one, which the readers reach after their reads
            float2 *pk = C.pk + (size_t)(team * 2 + (it & 1u)) * a.rows_max * RBQ;
            long long tk = tmg && t == 0 ? clock64() : 0;
            for (int base = 0; base < items * LPQ; base += TL) {
                const int idx = base + tl, item = idx / LPQ, sub = idx - item * LPQ;
                const bool act = item < items;
                const int rr = act ? item / C.RBQj : 0, qd = act ? item - rr * C.RBQj : 0, re = C.r0 + rr, be = t * 128 + re;
                const bool live = act && be < B;
                const int g0 = sub * NH, g1 = min(NGRP, g0 + NH);
                const uint32_t *fq = a.fx + ((((size_t)t * NGRP) * NKB + C.j) * RBQ + qd) * 512 + (size_t)re * 4;
                float4 fs = make_float4(0.f, 0.f, 0.f, 0.f);
                for (int ii0 = g0; ii0 < g1; ii0 += MMA_GB) {                       // group order (deterministic)
                    uint4 x[MMA_GB];
                    const int cnt = min(MMA_GB, g1 - ii0);
                    unsigned pend = live ? (1u << cnt) - 1u : 0u, spins = 0;
                    while (pend) {
#pragma unroll
                        for (int u = 0; u < MMA_GB; ++u)
                            if (pend >> u & 1) x[u] = ld_relaxed4(fq + (size_t)(ii0 + u) * fstride);
#pragma unroll
                        for (int u = 0; u < MMA_GB; ++u)
                            if ((pend >> u & 1) && tags_ok(x[u], tag)) pend &= ~(1u << u);
                        if (pend && (++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                    }
                    if (live) {
#pragma unroll
                        for (int u = 0; u < MMA_GB; ++u)
                            if (u < cnt) { fs.x += untag(x[u].x); fs.y += untag(x[u].y); fs.z += untag(x[u].z); fs.w += untag(x[u].w); }
                    }
                }
                if (tmg && t == 0 && base == 0) { const long long t_ = clock64(); tm[0] += t_ - tk; tk = t_; tmx += t_ - *reinterpret_cast<volatile long long *>(C.bars + MB_STAMP); mma_trace(a, C.c, n, 5); }
                // join the parts of the group range (fp32 addition is commutative: every lane of the quad gets the same bits)
                if (LPQ >= 2) {
                    fs.x += __shfl_xor_sync(FLOW_FULL, fs.x, 1); fs.y += __shfl_xor_sync(FLOW_FULL, fs.y, 1);
                    fs.z += __shfl_xor_sync(FLOW_FULL, fs.z, 1); fs.w += __shfl_xor_sync(FLOW_FULL, fs.w, 1);
                }
                if (LPQ >= 4) {
                    fs.x += __shfl_xor_sync(FLOW_FULL, fs.x, 2); fs.y += __shfl_xor_sync(FLOW_FULL, fs.y, 2);
                    fs.z += __shfl_xor_sync(FLOW_FULL, fs.z, 2); fs.w += __shfl_xor_sync(FLOW_FULL, fs.w, 2);
                }
                // a5 linear update of the lane's EPL elements (fp64, delta form).  Rows beyond the batch and the padding of the last
                // quad carry zero state and zero coefficients, so they need no special case; the rare extras (trajectory output,
                // external force, second-order start at n = 0) go through a separate uniform branch.
                float qn[EPL], po = 0.f, pn = 0.f;
                const int e0 = (rr * RBQ + qd) * 4 + sub * EPL;
                const double *cf = reinterpret_cast<const double *>(C.coef + (size_t)t * C.nel * 28);
                const float *cw = reinterpret_cast<const float *>(cf + 3 * C.nel);
                double qv[EPL], vv[EPL], ckv[EPL], ckq[EPL], cr[EPL];
#pragma unroll
                for (int h = 0; h < EPL; ++h) {
                    qv[h] = sq[e0 + h]; vv[h] = sv[e0 + h]; ckv[h] = cf[e0 + h]; ckq[h] = cf[C.nel + e0 + h]; cr[h] = cf[2 * C.nel + e0 + h];
                }
                constexpr bool extras = EXTRAS;
#pragma unroll
                for (int h = 0; h < EPL; ++h) {
                    const int hq = sub * EPL + h;
                    const double fd = (double)(hq == 0 ? fs.x : hq == 1 ? fs.y : hq == 2 ? fs.z : fs.w);
                    double fe = 0.0;
                    if (extras && live && 4 * qd + hq < C.nb) {
                        const int k = C.k0 + 4 * qd + hq;
                        const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
                        if (a.traj) a.traj[((size_t)be * a.n_steps + n) * a.n_q + a.kperm[k]] = qv[h];
                        if (n == 0 && a.auto_start) vv[h] = (cr[h] != 0.0) ? a.astart[co] * qv[h] + a.half_T2 * fd : 0.0;
                        if (a.fext) fe = (double)a.fext[(size_t)be * a.n_steps + n] * a.gain[(size_t)be * a.NQP + k];
                    }
                    vv[h] = fma(ckv[h], vv[h], fma(-ckq[h], qv[h], cr[h] * (fe - fd)));
                    qv[h] += vv[h];
                    qn[h] = (float)qv[h];
                    po = fmaf(cw[e0 + h], qn[h], po); pn = fmaf(qn[h], qn[h], pn);
                }
                if (act) {
#pragma unroll
                    for (int h = 0; h < EPL; ++h) { sq[e0 + h] = qv[h]; sv[e0 + h] = vv[h]; }
                }
                if (tmg && t == 0 && base == 0) { const long long t_ = clock64(); tm[3] += t_ - tk; tk = t_; }
                if (live) mma_publish(a, C, t, re, qd, sub * EPL, EPL, qn);
                if (LPQ >= 2) { po += __shfl_xor_sync(FLOW_FULL, po, 1); pn += __shfl_xor_sync(FLOW_FULL, pn, 1); }
                if (LPQ >= 4) { po += __shfl_xor_sync(FLOW_FULL, po, 2); pn += __shfl_xor_sync(FLOW_FULL, pn, 2); }
                if (act && sub == 0) pk[item] = make_float2(po, pn);
            }
            if (tmg && t == 0) { const long long t_ = clock64(); tm[1] += t_ - tk; tk = t_; mma_trace(a, C.c, n, 6); }
            bar_named(2 + team, TL);
            if (tl == 0) {
                if (C.j == 0) {            // warp W must have consumed the pickup partials of q^n before any owner may go on to q^{n+2}
                    unsigned spins = 0;
                    while (C.wdone[t] < n + 1) if ((++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 24))) { *C.s_abort = 1; break; }
                }
                set_flag(a.qflag + (((size_t)t * NKB + C.j) * NGRP + C.i) * MMA_FS, (unsigned)n + 2u);
            }
            if (tmg && t == 0) { const long long t_ = clock64(); tm[2] += t_ - tk; tk = t_; *reinterpret_cast<volatile long long *>(C.bars + MB_STAMP + 1) = t_; mma_trace(a, C.c, n, 7); }
            if (tl < C.rows) {                                 // pickup partial of q^{n+1} for row tl
                float o = 0.f, nr = 0.f;
                for (int qd = 0; qd < C.RBQj; ++qd) { const float2 x = pk[tl * C.RBQj + qd]; o += x.x; nr += x.y; }
                unsigned long long *pp = a.px + ((((size_t)((n + 1) & 1) * MT + t) * NKB + C.j) * 128 + C.r0 + tl) * 2;
                const unsigned long long ep = (unsigned long long)((unsigned)n + 2u) << 32;
                const unsigned long long w0 = ep | __float_as_uint(o), w1 = ep | __float_as_uint(nr);
                asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(pp), "l"(w0), "l"(w1) : "memory");
            }
        }
    }
}

template <int LPQ, bool TIMING>
__device__ __forceinline__ void mma_owner_team(const MmaArgs &a, const MmaCta &C, const int team, const int NTEAM, const int tl, const int TL)
{
    const int NGRP = a.NGRP, NKB = a.NKB, RBQ = a.RBQ, B = a.batch, MT = a.MT;
    const int items = C.rows * C.RBQj;
    constexpr int EPL = 4 / LPQ;                               // elements of a quad each of its lanes updates
    const bool tmg = TIMING && team == 0 && tl == 0;
    long long tm[4] = {0, 0, 0, 0};
    long long tmf = 0;
    unsigned it = 0;                                           // tile-steps this team has handled: pk buffer = it & 1
    // ---- owner state, publish q^0 and its pickup partials ----
    for (int t = team; t < MT; t += NTEAM, ++it) {
        double *sq = C.sq + (size_t)t * C.nel, *sv = C.sv + (size_t)t * C.nel;
        float2 *pk = C.pk + (size_t)(team * 2 + (it & 1u)) * a.rows_max * RBQ;
        for (int base = 0; base < items * LPQ; base += TL) {
            const int idx = base + tl, item = idx / LPQ, sub = idx - item * LPQ;
            const bool act = item < items;
            const int rr = act ? item / C.RBQj : 0, qd = act ? item - rr * C.RBQj : 0, re = C.r0 + rr, be = t * 128 + re;
            float qn[EPL], po = 0.f, pn = 0.f;
#pragma unroll
            for (int h = 0; h < EPL; ++h) {
                const int kk = 4 * qd + sub * EPL + h, k = C.k0 + kk, e = (rr * RBQ + qd) * 4 + sub * EPL + h;
                double q = 0.0, v = 0.0, kvv = 0.0, kqq = 0.0, rc = 0.0; float wk = 0.f;
                if (act && be < B && kk < C.nb) {
                    q = a.q0[(size_t)be * a.NQP + k]; v = a.v0[(size_t)be * a.NQP + k];
                    const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
                    kvv = a.kv[co]; kqq = a.kq[co]; rc = a.r[co]; wk = a.w[co];
                }
                if (act) {
                    sq[e] = q; sv[e] = v;
                    double *cf = reinterpret_cast<double *>(C.coef + (size_t)t * C.nel * 28);
                    cf[e] = kvv; cf[C.nel + e] = kqq; cf[2 * C.nel + e] = rc;
                    reinterpret_cast<float *>(cf + 3 * C.nel)[e] = wk;
                }
                qn[h] = (float)q;
                if (act && be < B && kk < C.nb) {
                    po = fmaf(a.w[(size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k], qn[h], po); pn = fmaf(qn[h], qn[h], pn);
                }
            }
            if (act) mma_publish(a, C, t, re, qd, sub * EPL, EPL, qn);
            if (LPQ >= 2) { po += __shfl_xor_sync(FLOW_FULL, po, 1); pn += __shfl_xor_sync(FLOW_FULL, pn, 1); }
            if (LPQ >= 4) { po += __shfl_xor_sync(FLOW_FULL, po, 2); pn += __shfl_xor_sync(FLOW_FULL, pn, 2); }
            if (act && sub == 0) pk[item] = make_float2(po, pn);
        }
        bar_named(2 + team, TL);
        if (tl == 0) set_flag(a.qflag + (((size_t)t * NKB + C.j) * NGRP + C.i) * MMA_FS, 1u);
        if (tl < C.rows) {                                     // pickup partial of q^0 for row tl: buffer 0, epoch 1
            float o = 0.f, nr = 0.f;
            for (int qd = 0; qd < C.RBQj; ++qd) { const float2 x = pk[tl * C.RBQj + qd]; o += x.x; nr += x.y; }
            unsigned long long *pp = a.px + (((size_t)t * NKB + C.j) * 128 + C.r0 + tl) * 2;
            const unsigned long long w0 = (1ull << 32) | __float_as_uint(o), w1 = (1ull << 32) | __float_as_uint(nr);
            asm volatile("st.relaxed.gpu.global.v2.b64 [%0], {%1, %2};" ::"l"(pp), "l"(w0), "l"(w1) : "memory");
        }
    }

    const bool extras = a.traj != nullptr || a.fext != nullptr;
    if (extras) mma_owner_steps<LPQ, TIMING, true>(a, C, team, NTEAM, tl, TL, 0, a.n_steps, it, tm, tmf);
    else {
        if (a.auto_start) mma_owner_steps<LPQ, TIMING, true>(a, C, team, NTEAM, tl, TL, 0, min(1, a.n_steps), it, tm, tmf);
        mma_owner_steps<LPQ, TIMING, false>(a, C, team, NTEAM, tl, TL, a.auto_start ? 1 : 0, a.n_steps, it, tm, tmf);
    }
    if (tmg) { for (int x = 0; x < 4; ++x) a.timing[(size_t)C.c * 16 + 8 + x] = tm[x]; a.timing[(size_t)C.c * 16 + 14] = tmf; }
}

// W: block-0 CTAs only.  out[b][n] = sum over the k blocks of the pickup partials of q^n (a1 pickup + a6 write-out); rows of this CTA.
__device__ __forceinline__ void mma_pickup_warp(const MmaArgs &a, const MmaCta &C, const int lane)
{
    const int NKB = a.NKB, MT = a.MT, B = a.batch;
    for (int n = 0; n < a.n_steps; ++n) {
        for (int t = 0; t < MT; ++t) {
            for (int rr = lane; rr < C.rows; rr += 32) {
                const int re = C.r0 + rr, be = t * 128 + re;
                if (be >= B) continue;
                const unsigned long long *pp = a.px + ((((size_t)(n & 1) * MT + t) * NKB) * 128 + re) * 2;
                float o = 0.f, nr = 0.f;
                for (int j = 0; j < NKB; ++j) {                 // block order (deterministic)
                    unsigned long long w0, w1;
                    unsigned spins = 0;
                    do {
                        asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(w0), "=l"(w1) : "l"(pp + (size_t)j * 256) : "memory");
                        if ((unsigned)(w0 >> 32) == (unsigned)n + 1u && (unsigned)(w1 >> 32) == (unsigned)n + 1u) break;
                        if ((++spins & 1023u) == 0 && (*C.s_abort || spins > (1u << 21))) { *C.s_abort = 1; break; }
                        __nanosleep(100);
                    } while (true);
                    o += __uint_as_float((unsigned)w0); nr += __uint_as_float((unsigned)w1);
                }
                a.out[(size_t)be * a.n_steps + n] = o;
                int *sb = C.sbad + t * a.rows_max + rr;
                if (*sb < 0 && !(isfinite(o) && isfinite(nr))) *sb = n;
            }
            __syncwarp();
            if (lane == 0) C.wdone[t] = n + 1;
        }
    }
    for (int t = 0; t < MT; ++t)
        for (int rr = lane; rr < C.rows; rr += 32)
            if (t * 128 + C.r0 + rr < B) a.first_bad[t * 128 + C.r0 + rr] = C.sbad[t * a.rows_max + rr];
}

template <bool TIMING>
__global__ void __launch_bounds__(MMA_THREADS, 1) vk_mma_kernel(const MmaArgs a)
{
    extern __shared__ __align__(128) unsigned char mma_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const MmaSmem L = mma_smem_layout(a.slab_bytes, a.MT, a.rows_max, a.RBQ, a.NSTG);
    MmaCta C;
    C.c = blockIdx.x; C.i = C.c / a.NKB; C.j = C.c - C.i * a.NKB;
    C.bars = reinterpret_cast<uint64_t *>(mma_smem + L.bars);
    uint32_t *tptr = reinterpret_cast<uint32_t *>(C.bars + MB_TPTR);
    C.s_abort = reinterpret_cast<volatile int *>(C.bars + MB_ABORT);
    int *tab = reinterpret_cast<int *>(mma_smem + L.bars + MMA_TAB_OFF);
    C.kl = tab; C.nmode = tab + 64; C.fb = tab + 72; C.blk = tab + 88;
    C.sq = reinterpret_cast<double *>(mma_smem + L.sq); C.sv = reinterpret_cast<double *>(mma_smem + L.sv);
    C.coef = mma_smem + L.coef;
    C.pk = reinterpret_cast<float2 *>(mma_smem + L.pk);
    C.sbad = reinterpret_cast<int *>(mma_smem + L.sbad);
    C.wdone = reinterpret_cast<volatile int *>(mma_smem + L.wdone);
    C.slab = mma_smem + L.slab; C.ring = mma_smem + L.ring; C.gex = mma_smem + L.gex;
    C.nel = (size_t)a.rows_max * a.RBQ * 4;

    if (tid == 0) {
        for (int s = 0; s < a.NSTG; ++s) { mbar_init(smem_u32(C.bars + MB_FULL + s), 1); mbar_init(smem_u32(C.bars + MB_EMPTY + s), 1); }
        for (int s = 0; s < 3; ++s) { mbar_init(smem_u32(C.bars + MB_ACCF + s), 1); mbar_init(smem_u32(C.bars + MB_ACCE + s), 128); }
        for (int t = 0; t < MMA_MT_MAX; ++t) mbar_init(smem_u32(C.bars + MB_QRDY + t), 1);
        for (int s = 0; s < 2; ++s) { mbar_init(smem_u32(C.bars + MB_RS + s), 1); mbar_init(smem_u32(C.bars + MB_AG + s), 1); }
        *C.s_abort = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int x = tid; x < a.MT * a.rows_max; x += blockDim.x) C.sbad[x] = -1;
    if (tid < MMA_MT_MAX) C.wdone[tid] = 0;
    for (int x = tid; x < 4096; x += blockDim.x) reinterpret_cast<float *>(C.gex)[x] = 0.f;
    if (tid < a.KCL && tid < 64) tab[tid] = a.klist[(size_t)C.c * a.KCL + tid];
    if (tid < MMA_NG_MAX_DEV) tab[64 + tid] = tid < a.NG ? a.nlist[C.i * a.NG + tid] : -1;
    if (tid < 16) tab[72 + tid] = a.fblk[(size_t)C.c * 16 + tid];
    if (tid < 3 * a.NKB && tid < 48) tab[88 + tid] = a.blk[tid];
    {   // H slab of this CTA: loaded once, resident for the whole run
        const uint4 *src = reinterpret_cast<const uint4 *>(a.slabs + (size_t)C.c * a.slab_bytes / 2);
        uint4 *dst = reinterpret_cast<uint4 *>(C.slab);
        for (int x = tid; x < a.slab_bytes / 16; x += blockDim.x) dst[x] = __ldg(src + x);
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tptr)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (a.CL) {   // the peers' mbarriers and exchange areas are set up before anybody stores into them
        asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    C.tbase = *tptr;
    C.k0 = C.blk[3 * C.j]; C.nb = C.blk[3 * C.j + 1]; C.koff = C.blk[3 * C.j + 2]; C.RBQj = (C.nb + 3) >> 2;
    C.NGa = 0;
    for (int u = 0; u < a.NG; ++u) C.NGa += C.nmode[u] >= 0;
    C.r0 = 128 * C.i / a.NGRP; C.rows = 128 * (C.i + 1) / a.NGRP - C.r0;
    C.KCA = a.kcnt[C.c];
    const int MT = a.MT, S = a.S, NSTG = a.NSTG;
    const int kc0 = C.i % C.KCA;                    // the CTAs that read the same chunks (same k block, other n groups) start at different ones:
                                                    // spreads the reads of one tile's operand over the L2 slices instead of hammering one chunk

    if (warp >= 8) {
        // ---------------- E: epilogue groups ----------------------------------------------------------
        asm volatile("setmaxnreg.inc.sync.aligned.u32 176;");
        const int r = (warp & 3) * 32 + lane;
        if (a.RBT <= 32) mma_epilogue_warpgroup<1, TIMING>(a, C, (warp - 8) >> 2, r, (warp & 3) * 32);
        else mma_epilogue_warpgroup<2, TIMING>(a, C, (warp - 8) >> 2, r, (warp & 3) * 32);
    } else if (warp >= 4) {
        // ---------------- O: owner teams ----------------------------------------------------------------
        asm volatile("setmaxnreg.dec.sync.aligned.u32 128;");
        const int NTEAM = MT >= 2 ? 2 : 1, TS = 4 / NTEAM;
        const int ow = warp - 4, team = ow / TS, tl = (ow - team * TS) * 32 + lane;
        if (a.LPQ == 1) mma_owner_team<1, TIMING>(a, C, team, NTEAM, tl, TS * 32);
        else if (a.LPQ == 2) mma_owner_team<2, TIMING>(a, C, team, NTEAM, tl, TS * 32);
        else mma_owner_team<4, TIMING>(a, C, team, NTEAM, tl, TS * 32);
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
        if (warp == 0) {
            // ---------------- P: wait for q^n of the tile's source blocks, stream its K chunks by TMA ----
            const uint32_t pfull0 = smem_u32(C.bars + MB_FULL), pempty0 = smem_u32(C.bars + MB_EMPTY), pring0 = smem_u32(C.ring);
            int psg = 0; unsigned pph = 1;                       // ring stage and the parity of its EMPTY phase to wait for
            const int fcnt = a.fcnt[C.c];
            const bool tmg = TIMING && lane == 0;
            long long tmp = 0, tmq = 0;
            for (int n = 0; n < a.n_steps; ++n)
                for (int t = 0; t < MT; ++t) {
                    const long long tk = tmg && t == 0 ? clock64() : 0;
                    poll_flag_list(a.qflag + (size_t)t * a.NKB * a.NGRP * MMA_FS, C.fb, fcnt, a.NGRP, lane, (unsigned)n + 1u, C.s_abort);
                    __syncwarp();
                    if (tmg && t == 0) { const long long t_ = clock64(); tmp += t_ - tk; if (n > 0) tmq += t_ - *reinterpret_cast<volatile long long *>(C.bars + MB_STAMP + 1); }
                    if (lane == 0) {
                        mbar_arrive(smem_u32(C.bars + MB_QRDY + t));
                        asm volatile("fence.proxy.async.global;" ::: "memory");
                        const unsigned char *qsrc = reinterpret_cast<const unsigned char *>(a.Qop) + (size_t)t * a.KC * 8192;
                        int x = kc0;                                                   // walk the chunks from a per-CTA offset
                        for (int xx = 0; xx < C.KCA; ++xx) {
                            mma_wait_fast(pempty0 + 8 * psg, pph, C.s_abort);
                            mbar_expect_tx(pfull0 + 8 * psg, 8192);
                            tma_bulk_g2s(pring0 + psg * 8192, qsrc + (size_t)C.kl[x] * 8192, 8192, pfull0 + 8 * psg);
                            if (++psg == NSTG) { psg = 0; pph ^= 1u; }
                            if (++x == C.KCA) x = 0;
                        }
                    }
                    __syncwarp();
                }
            if (tmg) { a.timing[(size_t)C.c * 16 + 12] = tmp; a.timing[(size_t)C.c * 16 + 15] = tmq; }
        } else if (warp == 1) {
            // ---------------- M: the MMAs of every tile, in order --------------------------------------------
            // The whole warp runs the (uniform) loop and one elected lane issues: inside a lane-0 branch ptxas wraps every tcgen05
            // instruction in an ELECT / R2UR / branch loop; no division and one add per descriptor in the chunk loop.
            {
                const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(a.NC >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
                const uint32_t full0 = smem_u32(C.bars + MB_FULL), empty0 = smem_u32(C.bars + MB_EMPTY);
                const uint64_t dQ0 = umma_desc(smem_u32(C.ring)), dH0 = umma_desc(smem_u32(C.slab));     // + (byte offset >> 4)
                const uint32_t hstep = (uint32_t)(2 * a.NC * 32) >> 4, hlo = (uint32_t)(a.NC * 32) >> 4;
                int sg = 0; unsigned ph = 0;
                unsigned uses[3] = {0u, 0u, 0u};
                const bool tmg = TIMING;
                long long tmm = 0;
                for (int n = 0; n < a.n_steps; ++n)
                    for (int t = 0; t < MT; ++t) {
                        const int slot = t % S;
                        const unsigned use = slot == 0 ? uses[0]++ : slot == 1 ? uses[1]++ : uses[2]++;
                        if (use > 0) mbar_wait(smem_u32(C.bars + MB_ACCE + slot), (use - 1u) & 1u, C.s_abort);   // the slot's last tile left it
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t td = C.tbase + (uint32_t)(slot * a.NC);
                        long long tk = 0;
                        int x = kc0;                                                   // position in the list = position in the slab
                        for (int xx = 0; xx < C.KCA; ++xx) {
                            mma_wait_fast(full0 + 8 * sg, ph, C.s_abort);
                            if (tmg && t == 0 && xx == 0) tk = clock64();
                            const uint64_t qhi = dQ0 + (uint64_t)(sg * (8192 >> 4)), hhi = dH0 + (uint64_t)((uint32_t)x * hstep);
                            if (mma_elect_one()) {
                                umma_bf16(td, qhi, hhi, idesc, xx > 0);
                                umma_bf16(td, qhi + (4096 >> 4), hhi, idesc, 1);
                                umma_bf16(td, qhi, hhi + hlo, idesc, 1);
                                umma_commit(empty0 + 8 * sg);                                             // ring slot free when these MMAs retire
                            }
                            if (++sg == NSTG) { sg = 0; ph ^= 1u; }
                            if (++x == C.KCA) x = 0;
                        }
                        if (mma_elect_one()) umma_commit(smem_u32(C.bars + MB_ACCF + slot));             // t of this tile complete
                        if (tmg && t == 0) tmm += clock64() - tk;
                    }
                if (tmg && lane == 0) a.timing[(size_t)C.c * 16 + 13] = tmm;
            }
        } else if (warp == 2 && C.j == 0) {
            mma_pickup_warp(a, C, lane);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (a.CL) {   // no CTA of the cluster leaves while a peer may still store into its shared memory
        asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    if (tid == 0 && *C.s_abort) *a.timeout_flag = 1;
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(C.tbase), "r"(512));
}

}  // namespace modal_dev
