// vk_mma.cuh -- batched MODAL_VK time loop on tcgen05 tensor cores, ONE persistent sm_100a kernel
// (layout in mma_schedule.hpp).
//
// Per time step, for up to 256 samples at once (two M tiles of 128):
//   t[b][(n,k)] = sum_r q[b][r] H^n[k][r]        tcgen05.mma kind::f16, bf16 hi/lo split, 3 MMAs per K chunk,
//                                                A = q chunk streamed by TMA from L2, B = H slab resident in
//                                                shared memory, D = t in TMEM (fp32), kept for both epilogues
//   G[b][n]  = sum_k q[b][k] t[b][(n,k)]         epilogue 1 (tcgen05.ld, one thread per sample), partial over
//                                                the CTA's 16 rows k; summed over the k blocks through L2
//   eta      = s_n[b] G[b][n]                    (Eq. 9, C eliminated by PAPER.md:283)
//   f[b][k]  = sum_n eta[b][n] t[b][(n,k)]       epilogue 2, partial over the CTA's modes n; summed over
//                                                the n groups through L2 by the owner of (b, k)
//   fp64 delta-form update of the owner's (q, v) (Eq. 19-23), q republished as fp32 and
//   as bf16 hi/lo in operand layout; pickup out[b][n] = w . q^n.
// CTA (i,j) owns in-plane modes of group i and rows k of block j.  CTAs synchronise with epoch
// flags in global memory (writer: stores, fence, flag; reader: acquire flag, L2 loads): no grid barrier.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_flow.cuh"   // mbarrier / TMA / bounded-wait helpers

namespace modal_dev {

constexpr int MMA_NSTG = 6;          // q-operand ring stages (8 KiB each: 128 rows x 16 K x hi/lo)
constexpr int MMA_THREADS = 320;     // warp 0 TMA producer, 1 MMA issuer, 2-5 / 6-9 epilogue + pickup of tile 0 / 1 (<= 204 registers)

struct MmaArgs {
    const uint16_t *slabs;      // [G][slab_bytes] bf16 hi/lo operand slabs of H
    int slab_bytes;
    int NKB, NGRP, NG, NGP, NC, KC, KP, G;
    const int *n0;              // [NGRP+1]
    int n_q, n_phi, NQP;
    int batch, n_steps, MT;     // batch <= 256; MT = M tiles in use
    int coeff_stride_q, coeff_stride_phi;
    const double *kv, *kq, *r, *astart;
    const float *s, *w;
    const double *q0, *v0;
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; int *first_bad;
    // exchange (global, L2 resident)
    uint16_t *Qg;               // [2][KC][2][4096 B]  q as bf16 hi/lo operand chunks
    float *qf;                  // [256][KP]           q fp32
    float *Gx;                  // [G][2][128][NGP]    partial G
    float *fx;                  // [NGRP][2][128][KP]  partial f
    unsigned *gflag, *fflag, *qflag;   // [G][2] epochs
    long long *timing;          // optional [G][8] cycle counters of tile 0 (MODAL_FLOW_TIMING)
};

__device__ __forceinline__ void poll_flag(const unsigned *p, unsigned epoch, volatile int *abortp)
{
    unsigned v, spins = 0;
    do {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
        if (v >= epoch) break;
        if ((++spins & 1023u) == 0 && (*abortp || spins > (1u << 21))) { *abortp = 1; flow_timeout_flag = 1; break; }
    } while (true);
}
__device__ __forceinline__ void set_flag(unsigned *p, unsigned epoch)
{
    __threadfence();
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
// flags p[idx * stride], idx = first, first + 32, ... < count: all loads of a lane in flight together
__device__ __forceinline__ void poll_flags_strided(const unsigned *p, int stride, int first, int count, unsigned epoch,
                                                   volatile int *abortp)
{
    for (int base = first; base < count; base += 256) {
        unsigned pend = 0, spins = 0;
#pragma unroll
        for (int u = 0; u < 8; ++u) if (base + 32 * u < count) pend |= 1u << u;
        while (pend) {
            unsigned v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (pend >> u & 1) asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v[u]) : "l"(p + (size_t)(base + 32 * u) * stride) : "memory");
#pragma unroll
            for (int u = 0; u < 8; ++u) if ((pend >> u & 1) && v[u] >= epoch) pend &= ~(1u << u);
            if (pend && (++spins & 1023u) == 0 && (*abortp || spins > (1u << 21))) { *abortp = 1; flow_timeout_flag = 1; break; }
        }
    }
}
__device__ __forceinline__ uint16_t bf16_rn_dev(float x)
{
    uint32_t u = __float_as_uint(x);
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

struct MmaSmem { size_t bars, sq, sv, sbad, cst, slab, ring, total; };
__host__ __device__ inline int mma_nel_max(int NGRP) { return ((128 + NGRP - 1) / NGRP + 1) * 16; }
__host__ __device__ inline MmaSmem mma_smem_layout(int slab_bytes, int NGRP)
{
    MmaSmem L; size_t o = 0;
    const size_t nel = (size_t)mma_nel_max(NGRP);
    L.bars = o; o += 256;                                  // mbarriers, tmem pointer, abort word
    L.sq = o;   o += 2 * nel * 8;                          // owner state q [2 tiles][nel]
    L.sv = o;   o += 2 * nel * 8;
    L.sbad = o; o += 256 * 4;
    L.cst = o;  o += 256 * 128;                            // per epilogue thread: s_n[16] floats + 8 doubles of update coefficients
    o = flow_align(o, 128);
    L.slab = o; o += (size_t)slab_bytes;
    o = flow_align(o, 128);
    L.ring = o; o += (size_t)MMA_NSTG * 8192;
    L.total = o;
    return L;
}

// One epilogue group = 128 threads = one M tile of 128 samples (thread <-> TMEM lane <-> sample).
__device__ __forceinline__ void mma_epilogue_group(const MmaArgs &a, const int mt, const int c, const int i, const int j,
                                                   const int r, uint64_t *bars, double *sq, double *sv,
                                                   const uint32_t tbase, volatile int *s_abort, const int lane_base,
                                                   int *sbad, const int gw, const int lane, unsigned char *cst)
{
    const int NC = a.NC, NG = a.NG, NGP = a.NGP, KP = a.KP, NKB = a.NKB, NGRP = a.NGRP, B = a.batch;
    const int b = mt * 128 + r;
    const bool valid = b < B;
    const int bar_id = 2 + mt;
    const int n0 = a.n0[i];
    const size_t cq = (size_t)(a.coeff_stride_q ? (valid ? b : 0) : 0) * a.NQP;
    const float *sb = a.s + (size_t)(a.coeff_stride_phi ? (valid ? b : 0) : 0) * a.n_phi;
    // the (sample, k) elements this group owns for the update: rows r0..r1 of the tile, 16 modes of block j
    const int r0 = 128 * i / NGRP, r1 = 128 * (i + 1) / NGRP, nel = (r1 - r0) * 16;
    uint16_t *Qt = a.Qg + (size_t)mt * a.KC * 8192 / 2 + (size_t)j * 8192 / 2;     // chunk kc = j of this tile (hi; lo at +4096 B)
    // ---- publish q^0 ----
    for (int e = r; e < nel; e += 128) {
        const int re = r0 + (e >> 4), kk = e & 15, be = mt * 128 + re, k = j * 16 + kk;
        double q = 0.0, v = 0.0;
        if (be < B) { q = a.q0[(size_t)be * a.NQP + k]; v = a.v0[(size_t)be * a.NQP + k]; }
        sq[e] = q; sv[e] = v;
        if (be < B) {
            const float qfl = (float)q;
            a.qf[(size_t)be * KP + k] = qfl;
            const uint16_t hi = bf16_rn_dev(qfl), lo = bf16_rn_dev(qfl - __uint_as_float((uint32_t)hi << 16));
            const int off = ((re >> 3) * 256 + (kk >> 3) * 128 + (re & 7) * 16 + (kk & 7) * 2) >> 1;
            Qt[off] = hi; Qt[2048 + off] = lo;
        }
    }
    bar_named(bar_id, 128);
    if (r == 0) set_flag(a.qflag + c * 2 + mt, 1u);

    // per-thread constants, loaded once: __threadfence (gpu scope) invalidates L1, so anything re-read from
    // global inside the step loop would pay an L2 round trip every time
    float *sreg = reinterpret_cast<float *>(cst);                                // [16] s_n of this sample
    double *ccf = reinterpret_cast<double *>(cst + 64);                         // [2][4] kv, kq, r, astart of the owned elements
    for (int u = 0; u < 16; ++u) sreg[u] = (u < NG && n0 + u < a.n_phi) ? sb[n0 + u] : 0.f;
    const bool fast = nel <= 256;                                               // <= 2 owned elements per thread
    if (fast)
        for (int h = 0; h < 2; ++h) {
            const int e = r + 128 * h;
            ccf[4 * h] = ccf[4 * h + 1] = ccf[4 * h + 2] = ccf[4 * h + 3] = 0.0;
            if (e < nel) {
                const int re = r0 + (e >> 4), be = mt * 128 + re, k = j * 16 + (e & 15);
                if (be < B) {
                    const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
                    ccf[4 * h] = a.kv[co]; ccf[4 * h + 1] = a.kq[co]; ccf[4 * h + 2] = a.r[co]; ccf[4 * h + 3] = a.astart[co];
                }
            }
        }
    const uint32_t taddr0 = tbase + ((uint32_t)lane_base << 16) + (uint32_t)(mt * NC);
    const bool tmg = a.timing && r == 0 && mt == 0;
    long long *tm = a.timing + (size_t)c * 8;
    for (int n = 0; n < a.n_steps; ++n) {
        const unsigned ep = (unsigned)n + 1u;
        long long tk = tmg ? clock64() : 0;
        mbar_wait(smem_u32(bars + 16 + mt), n & 1, s_abort);                       // q^n published by everybody
        if (tmg) { const long long t_ = clock64(); tm[0] += t_ - tk; tk = t_; }
        // ---- a1 pickup + a6 write-out: out[b][n] = w . q^n for the samples b = c, c+G, ... of this tile ----
        for (int m = gw, b2 = c + gw * a.G; b2 < B; m += 4, b2 += 4 * a.G) {
            if (b2 / 128 != mt) continue;
            const float *wb = a.w + (size_t)(a.coeff_stride_q ? b2 : 0) * a.NQP;
            float o = 0.f, nrm = 0.f;
            for (int k = lane; k < a.n_q; k += 32) {
                const float qk = __ldcg(a.qf + (size_t)b2 * KP + k);
                o = fmaf(wb[k], qk, o); nrm = fmaf(qk, qk, nrm);
            }
#pragma unroll
            for (int sh = 16; sh >= 1; sh >>= 1) { o += __shfl_xor_sync(FLOW_FULL, o, sh); nrm += __shfl_xor_sync(FLOW_FULL, nrm, sh); }
            if (lane == 0) {
                a.out[(size_t)b2 * a.n_steps + n] = o;
                if (sbad[m] < 0 && !(isfinite(o) && isfinite(nrm))) sbad[m] = n;
            }
        }
        float q16[16];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
            if (valid) x = __ldcg(reinterpret_cast<const float4 *>(a.qf + (size_t)b * KP + j * 16) + u);
            q16[4 * u] = x.x; q16[4 * u + 1] = x.y; q16[4 * u + 2] = x.z; q16[4 * u + 3] = x.w;
        }
        mbar_wait(smem_u32(bars + 12 + mt), n & 1, s_abort);                       // t of this tile is in TMEM
        if (tmg) { const long long t_ = clock64(); tm[1] += t_ - tk; tk = t_; }
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // ---- epilogue 1: partial G over the 16 rows k of block j ----
        float4 *gout = reinterpret_cast<float4 *>(a.Gx + ((size_t)(c * 2 + mt) * 128 + r) * NGP);
        for (int n4 = 0; n4 < NGP / 4; ++n4) {
            float g4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int h = 0; h < 2; ++h) {                                       // two modes per TMEM wait
                const int nl = n4 * 4 + 2 * h;
                uint32_t v0[16], v1[16];
                if (nl < NG) tmem_ld16_nowait(taddr0 + nl * 16, v0);
                if (nl + 1 < NG) tmem_ld16_nowait(taddr0 + (nl + 1) * 16, v1);
                tmem_ld_wait();
#pragma unroll
                for (int kk = 0; kk < 16; ++kk) {
                    if (nl < NG) g4[2 * h] = fmaf(q16[kk], __uint_as_float(v0[kk]), g4[2 * h]);
                    if (nl + 1 < NG) g4[2 * h + 1] = fmaf(q16[kk], __uint_as_float(v1[kk]), g4[2 * h + 1]);
                }
            }
            gout[n4] = make_float4(g4[0], g4[1], g4[2], g4[3]);
        }
        bar_named(bar_id, 128);
        if (r == 0) set_flag(a.gflag + c * 2 + mt, ep);
        if (tmg) { const long long t_ = clock64(); tm[2] += t_ - tk; tk = t_; }
        if (r < 32) poll_flags_strided(a.gflag + (i * NKB) * 2 + mt, 2, r, NKB, ep, s_abort);
        bar_named(bar_id, 128);
        if (tmg) { const long long t_ = clock64(); tm[3] += t_ - tk; tk = t_; }
        float eta[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) eta[u] = 0.f;
        {   // sum over the k blocks in fixed order (deterministic); 8 partial rows in flight per batch
            const float4 *gp0 = reinterpret_cast<const float4 *>(a.Gx + ((size_t)((i * NKB) * 2 + mt) * 128 + r) * NGP);
            const size_t gstride = (size_t)2 * 128 * NGP / 4;                       // float4 between consecutive k blocks
#pragma unroll
            for (int n4 = 0; n4 < 4; ++n4)
                if (n4 < NGP / 4)
                    for (int jj0 = 0; jj0 < NKB; jj0 += 8) {
                        float4 x[8];
#pragma unroll
                        for (int u = 0; u < 8; ++u) if (jj0 + u < NKB) x[u] = __ldcg(gp0 + (size_t)(jj0 + u) * gstride + n4);
#pragma unroll
                        for (int u = 0; u < 8; ++u)
                            if (jj0 + u < NKB) { eta[4 * n4] += x[u].x; eta[4 * n4 + 1] += x[u].y; eta[4 * n4 + 2] += x[u].z; eta[4 * n4 + 3] += x[u].w; }
                    }
        }
#pragma unroll
        for (int u = 0; u < 16; ++u) eta[u] *= sreg[u];                             // eta_n = s_n G_n
        if (tmg) { const long long t_ = clock64(); tm[7] += t_ - tk; tk = t_; }
        // ---- epilogue 2: partial force over the modes n of group i ----
        float facc[16];
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) facc[kk] = 0.f;
#pragma unroll
        for (int nl = 0; nl < 16; nl += 2)
            if (nl < NG) {
                uint32_t v0[16], v1[16];
                tmem_ld16_nowait(taddr0 + nl * 16, v0);
                if (nl + 1 < NG) tmem_ld16_nowait(taddr0 + (nl + 1) * 16, v1);
                tmem_ld_wait();
#pragma unroll
                for (int kk = 0; kk < 16; ++kk) {
                    facc[kk] = fmaf(eta[nl], __uint_as_float(v0[kk]), facc[kk]);
                    if (nl + 1 < NG) facc[kk] = fmaf(eta[nl + 1], __uint_as_float(v1[kk]), facc[kk]);
                }
            }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        mbar_arrive(smem_u32(bars + 14 + mt));                                      // TMEM tile may be overwritten
        float4 *fout = reinterpret_cast<float4 *>(a.fx + ((size_t)(i * 2 + mt) * 128 + r) * KP + j * 16);
#pragma unroll
        for (int u = 0; u < 4; ++u) fout[u] = make_float4(facc[4 * u], facc[4 * u + 1], facc[4 * u + 2], facc[4 * u + 3]);
        bar_named(bar_id, 128);
        if (r == 0) set_flag(a.fflag + c * 2 + mt, ep);
        if (tmg) { const long long t_ = clock64(); tm[4] += t_ - tk; tk = t_; }
        if (r < 32) poll_flags_strided(a.fflag + j * 2 + mt, 2 * NKB, r, NGRP, ep, s_abort);
        bar_named(bar_id, 128);
        if (tmg) { const long long t_ = clock64(); tm[5] += t_ - tk; tk = t_; }
        // ---- owner update: group-ordered sum of the partial forces, a5 linear update (fp64, delta form) ----
        for (int e = r; e < nel; e += 128) {
            const int re = r0 + (e >> 4), kk = e & 15, be = mt * 128 + re, k = j * 16 + kk;
            if (be >= B) continue;
            float f = 0.f;
            {
                const float *fp0 = a.fx + ((size_t)mt * 128 + re) * KP + k;
                const size_t fstride = (size_t)2 * 128 * KP;
                for (int ii0 = 0; ii0 < NGRP; ii0 += 16) {                          // group order; 16 loads in flight
                    float x[16];
#pragma unroll
                    for (int u = 0; u < 16; ++u) if (ii0 + u < NGRP) x[u] = __ldcg(fp0 + (size_t)(ii0 + u) * fstride);
#pragma unroll
                    for (int u = 0; u < 16; ++u) if (ii0 + u < NGRP) f += x[u];
                }
            }
            const size_t co = (size_t)(a.coeff_stride_q ? be : 0) * a.NQP + k;
            const int h = e >= 128 ? 1 : 0;
            const double fd = (double)f;
            const double rr = fast ? ccf[4 * h + 2] : a.r[co], kvv = fast ? ccf[4 * h] : a.kv[co], kqq = fast ? ccf[4 * h + 1] : a.kq[co];
            double q = sq[e], v = sv[e];
            if (a.traj && k < a.n_q) a.traj[((size_t)be * a.n_steps + n) * a.n_q + k] = q;
            if (n == 0 && a.auto_start) v = (rr != 0.0) ? (fast ? ccf[4 * h + 3] : a.astart[co]) * q + a.half_T2 * fd : 0.0;
            const double fe = a.fext ? (double)a.fext[(size_t)be * a.n_steps + n] * a.gain[(size_t)be * a.NQP + k] : 0.0;
            v = kvv * v - kqq * q + rr * (fe - fd);
            q += v;
            sq[e] = q; sv[e] = v;
            const float qfl = (float)q;
            a.qf[(size_t)be * KP + k] = qfl;
            const uint16_t hi = bf16_rn_dev(qfl), lo = bf16_rn_dev(qfl - __uint_as_float((uint32_t)hi << 16));
            const int off = ((re >> 3) * 256 + (kk >> 3) * 128 + (re & 7) * 16 + (kk & 7) * 2) >> 1;
            Qt[off] = hi; Qt[2048 + off] = lo;
        }
        bar_named(bar_id, 128);
        if (r == 0) set_flag(a.qflag + c * 2 + mt, ep + 1u);
        if (tmg) { const long long t_ = clock64(); tm[6] += t_ - tk; tk = t_; }
    }
    if (lane == 0)
        for (int m = gw, b2 = c + gw * a.G; b2 < B; m += 4, b2 += 4 * a.G)
            if (b2 / 128 == mt) a.first_bad[b2] = sbad[m];
    (void)cq;
}

__global__ void __launch_bounds__(MMA_THREADS, 1) vk_mma_kernel(const MmaArgs a)
{
    extern __shared__ __align__(128) unsigned char mma_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x, i = c / a.NKB, j = c - i * a.NKB;
    const MmaSmem L = mma_smem_layout(a.slab_bytes, a.NGRP);
    uint64_t *bars = reinterpret_cast<uint64_t *>(mma_smem + L.bars);      // full[0..5] empty[6..11] acc_full[12,13]
    uint32_t *tptr = reinterpret_cast<uint32_t *>(bars + 20);              // acc_empty[14,15] qready[16,17] pick_done[18]
    volatile int *s_abort = reinterpret_cast<volatile int *>(bars + 21);
    double *sq = reinterpret_cast<double *>(mma_smem + L.sq), *sv = reinterpret_cast<double *>(mma_smem + L.sv);
    int *sbad = reinterpret_cast<int *>(mma_smem + L.sbad);
    unsigned char *cst = mma_smem + L.cst;
    unsigned char *slab = mma_smem + L.slab, *ring = mma_smem + L.ring;
    const int nel_max = mma_nel_max(a.NGRP);

    if (tid == 0) {
        for (int s = 0; s < MMA_NSTG; ++s) { mbar_init(smem_u32(bars + s), 1); mbar_init(smem_u32(bars + 6 + s), 1); }
        for (int m = 0; m < 2; ++m) {
            mbar_init(smem_u32(bars + 12 + m), 1); mbar_init(smem_u32(bars + 14 + m), 128); mbar_init(smem_u32(bars + 16 + m), 1);
        }
        mbar_init(smem_u32(bars + 18), 2);
        *s_abort = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int x = tid; x < 256; x += blockDim.x) sbad[x] = -1;
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

    if (warp == 0) {
        // ---------------- producer: wait for q^n of a tile, stream it through the ring by TMA ----------
        int stage = 0; unsigned ph = 0;
        for (int n = 0; n < a.n_steps; ++n)
            for (int mt = 0; mt < MT; ++mt) {
                poll_flags_strided(a.qflag + mt, 2, lane, a.G, (unsigned)n + 1u, s_abort);
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(smem_u32(bars + 16 + mt));
                    asm volatile("fence.proxy.async.global;" ::: "memory");
                    for (int kc = 0; kc < KC; ++kc) {
                        mbar_wait(smem_u32(bars + 6 + stage), ph ^ 1, s_abort);
                        mbar_expect_tx(smem_u32(bars + stage), 8192);
                        tma_bulk_g2s(smem_u32(ring + stage * 8192), a.Qg + ((size_t)mt * KC + kc) * 4096, 8192, smem_u32(bars + stage));
                        if (++stage == MMA_NSTG) { stage = 0; ph ^= 1; }
                    }
                }
                __syncwarp();
            }
    } else if (warp == 1) {
        // ---------------- MMA issuer: one thread --------------------------------------------------------
        if (lane == 0) {
            const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(NC >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
            int stage = 0; unsigned ph = 0;
            for (int n = 0; n < a.n_steps; ++n)
                for (int mt = 0; mt < MT; ++mt) {
                    mbar_wait(smem_u32(bars + 14 + mt), (n & 1) ^ 1, s_abort);              // epilogues of step n-1 left the tile
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t td = tbase + (uint32_t)(mt * NC);
                    for (int kc = 0; kc < KC; ++kc) {
                        mbar_wait(smem_u32(bars + stage), ph, s_abort);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t qa = smem_u32(ring + stage * 8192), hb = smem_u32(slab + (size_t)kc * 2 * NC * 32);
                        const uint64_t qhi = umma_desc(qa), qlo = umma_desc(qa + 4096);
                        const uint64_t hhi = umma_desc(hb), hlo = umma_desc(hb + NC * 32);
                        umma_bf16(td, qhi, hhi, idesc, kc > 0);
                        umma_bf16(td, qlo, hhi, idesc, 1);
                        umma_bf16(td, qhi, hlo, idesc, 1);
                        umma_commit(smem_u32(bars + 6 + stage));                           // ring slot free when these MMAs retire
                        if (++stage == MMA_NSTG) { stage = 0; ph ^= 1; }
                    }
                    umma_commit(smem_u32(bars + 12 + mt));                                 // t of tile mt complete
                }
        }
    } else {
        const int mt = (warp - 2) >> 2, gw = (warp - 2) & 3;
        if (mt < MT)
            mma_epilogue_group(a, mt, c, i, j, (warp & 3) * 32 + lane, bars, sq + (size_t)mt * nel_max, sv + (size_t)mt * nel_max,
                               tbase, s_abort, (warp & 3) * 32, sbad, gw, lane, cst + (size_t)(tid - 64) * 128);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tbase), "r"(512));
}

}  // namespace modal_dev
