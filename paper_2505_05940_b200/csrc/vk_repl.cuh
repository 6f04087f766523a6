// vk_repl.cuh -- von Karman time loop of ONE sample of a LARGE plate (C4: N_q = 400, N_phi = 200; BASELINE.json configs[1], the
// headline) with replicated state and ONE cross-CTA hop through L2 per time step.  Layout: repl_schedule.hpp.  DESIGN.md 7.9.
//
// vk_flow_kernel spreads the tiles of H over the CTAs and pays two L2 hops per step (partial forces -> owners, new state ->
// everybody), 8.75 us per step at C4 of which the contraction is a third.  Here every CTA keeps the WHOLE fp64 state (thread k <->
// mode k, bit-identical replicas) and owns whole in-plane modes n, whose H^n sits in shared memory as the dense blocks of its
// parity structure (a <= b only: H^n is symmetric):
//   t_n = H^n q            every thread one item = (block, chunk of rows, quad of columns): float4 loads, column sums in registers,
//                          row sums per row to shared memory; thread k then joins the partials of mode k          (a2)
//   G_n = q . t_n, eta_n = s_n G_n, f += eta_n t_n   block sums, all local                                         (a3, a4)
//   exchange: the CTA's partial force (N_q floats) is reduce-scattered inside its thread-block cluster through distributed shared
//             memory (st.async + complete_tx), the cluster's sums go to L2 as tagged 64-bit words {fp32, epoch}, double-buffered by
//             step parity, and every CTA gathers the sums of all clusters (pairs of modes per 16-byte load, all loads of a round
//             in flight, fixed order)
//   v <- kv v - kq q + r (fext - f),  q <- q + v     fp64, every CTA the same                                     (a5)
//   out[n] = w . q^n       by the CTA `out_cta`                                                                    (a1, a6)
// (Eq. 9-11 with C eliminated; Eq. 19/20 in delta form.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_mma.cuh"   // mbarrier / distributed shared memory helpers, st_tag

namespace modal_dev {

constexpr int RP_THREADS = 512, RP_MAXM = 4, RP_MAXCLS = 8, RP_HDR = 16, RP_ITEM = 8, RP_JOIN = 4;
constexpr int RP_CTA_STRIDE = RP_HDR + RP_THREADS * RP_ITEM + RP_MAXM * RP_MAXCLS * RP_JOIN;
constexpr int RP_CL_MAX = 8;            // CTAs of a cluster
constexpr int RP_GROUND = 9;            // 16-byte loads of one gather round in flight per thread
constexpr int RP_NSUB_MAX = 4;          // gather sub-groups

struct ReplArgs {
    int n_q, NQ2, n_phi, NQP, n_steps, G, CL, NCL, SL, out_cta;
    int hfloats_max, cp_max, rp_max;
    const float *Hp; const int *tab; const int *cls;      // cls: [n_q] class of internal mode k
    const double *kv, *kq, *r, *astart;
    const float *s, *w;
    const double *q0, *v0;
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; const int *kperm; int *first_bad;
    unsigned long long *X;               // [2][NCL][NQ2] tagged words
    int *timeout_flag;
    long long *timing;                   // optional [G][8]
};

__host__ __device__ inline size_t repl_smem_bytes(int hfloats_max, int cp_max, int rp_max, int CL, int SL)
{
    return ((size_t)hfloats_max + cp_max + rp_max + 4 + (size_t)2 * CL * SL) * 4 + 64;
}

// sums of the first NV (<= 8) values over the block; every thread gets the same bits.  red: [16 warps][8] floats of THIS step's parity
// (the caller double-buffers, so one barrier is enough: the buffer is rewritten two steps later, behind several barriers).
// Level-major butterflies (the NV shuffles of a level are independent), then lane y of every warp reads the row of warp y and a
// 16-lane butterfly joins them: 16 dependent shared-memory loads per thread measured 640 cycles here, this 150.
template <int NV>
__device__ __forceinline__ void rp_block_sum(float (&a)[8], float *red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
#pragma unroll
        for (int x = 0; x < NV; ++x) a[x] += __shfl_xor_sync(0xffffffffu, a[x], m);
    }
    if (lane == 0) {
        *reinterpret_cast<float4 *>(red + warp * 8) = make_float4(a[0], a[1], a[2], a[3]);
        if (NV > 4) *reinterpret_cast<float4 *>(red + warp * 8 + 4) = make_float4(a[4], a[5], a[6], a[7]);
    }
    __syncthreads();
    const float4 u = *reinterpret_cast<const float4 *>(red + (lane & 15) * 8);
    a[0] = u.x; a[1] = u.y; a[2] = u.z; a[3] = u.w;
    if (NV > 4) {
        const float4 w = *reinterpret_cast<const float4 *>(red + (lane & 15) * 8 + 4);
        a[4] = w.x; a[5] = w.y; a[6] = w.z; a[7] = w.w;
    }
#pragma unroll
    for (int m = 8; m >= 1; m >>= 1) {
#pragma unroll
        for (int x = 0; x < NV; ++x) a[x] += __shfl_xor_sync(0xffffffffu, a[x], m);
    }
}

// MM: mode slots the instance carries (2 when no CTA holds more than two in-plane modes, as at C4: half the unrolled join code)
template <bool TIMING, int MM = RP_MAXM>
__global__ void __launch_bounds__(RP_THREADS, 1) vk_repl_kernel(const ReplArgs a)
{
    __shared__ __align__(16) float qs[RP_THREADS + 8];
    __shared__ __align__(16) float red[2 * 16 * 8];
    __shared__ __align__(16) float part2[RP_NSUB_MAX * RP_THREADS];     // partial sums of the gather sub-groups
    __shared__ __align__(8) uint64_t rsbar[2];
    __shared__ volatile int s_abort;
    extern __shared__ __align__(16) float rp_smem[];
    float *Hs = rp_smem;                                       // the CTA's blocks
    float *cpart = Hs + a.hfloats_max;
    float *rpart = cpart + a.cp_max;
    float *rs = rpart + a.rp_max + 4;                          // [2][CL][SL] reduce-scatter landing zone
    const int k = threadIdx.x, g = blockIdx.x;
    const int *T = a.tab + (size_t)g * RP_CTA_STRIDE;
    const int nmodes = T[2];
    uint32_t rank = 0, cid = g;
    if (a.CL > 1) { asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank)); cid = g / a.CL; }
    // item of this thread, join descriptors of mode k
    const int4 I0 = *reinterpret_cast<const int4 *>(T + RP_HDR + k * RP_ITEM), I1 = *reinterpret_cast<const int4 *>(T + RP_HDR + k * RP_ITEM + 4);
    const bool has_item = k < T[3];
    const bool mine = k < a.n_q;
    int4 J[MM];
    {
        const int c = mine ? a.cls[k] : 0, c0 = mine ? k : 0;
        int first = c0;                                        // first mode of the class: walk down while the class is the same
        while (first > 0 && a.cls[first - 1] == c) --first;
#pragma unroll
        for (int m = 0; m < MM; ++m) {
            J[m] = make_int4(0, 0, 0, 0);
            if (mine && m < nmodes) {
                J[m] = *reinterpret_cast<const int4 *>(T + RP_HDR + RP_THREADS * RP_ITEM + (m * RP_MAXCLS + c) * RP_JOIN);
                if (J[m].x == 2) { J[m].y += (k - first) * J[m].w; J[m].w = 1; }      // row sums: the row's quads are consecutive (odd row pitch)
                else J[m].y += k - first;                                              // column sums: one partial per chunk of rows
            }
        }
    }
    float sm_[MM];
#pragma unroll
    for (int m = 0; m < MM; ++m) sm_[m] = m < nmodes ? a.s[T[4 + m]] : 0.f;
    double q = 0.0, v = 0.0, kv = 0.0, kq = 0.0, r = 0.0, ast = 0.0, gn = 0.0; float wk = 0.f;
    if (mine) {
        q = a.q0[k]; v = a.v0[k]; kv = a.kv[k]; kq = a.kq[k]; r = a.r[k]; ast = a.astart[k]; wk = a.w[k];
        if (a.fext) gn = a.gain[k];
    }
    if (k == 0) {
        s_abort = 0;
        mbar_init(smem_u32(&rsbar[0]), 1); mbar_init(smem_u32(&rsbar[1]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        const float4 *src = reinterpret_cast<const float4 *>(a.Hp) + T[0];
        float4 *dst = reinterpret_cast<float4 *>(Hs);
        for (int i = k; i < T[1] / 4; i += RP_THREADS) dst[i] = __ldg(src + i);
    }
    if (k < 8) qs[RP_THREADS + k] = 0.f;
    // reduce-scatter targets: mode k goes to rank k / SL of the cluster
    const int SL = a.SL, CL = a.CL;
    const bool xk = k < a.NQ2;                                 // the exchange runs over NQ2 = N_q rounded up to even (pairs)
    const int jt = xk ? k / SL : 0;
    uint32_t rs_remote = 0, bar_remote = 0;
    if (CL > 1) {
        rs_remote = dsm_map(smem_u32(rs + (size_t)rank * SL + (k - jt * SL)), (uint32_t)jt);
        bar_remote = dsm_map(smem_u32(&rsbar[0]), (uint32_t)jt);
    }
    const int my0 = (int)rank * SL, mylen = max(0, min(a.NQ2, my0 + SL) - my0);
    // gather: pairs of modes per 16-byte load; sub-groups of threads share the clusters
    const int NP = a.NQ2 >> 1;
    const int NSUB = min(RP_THREADS / NP, RP_NSUB_MAX);
    const int sub = k / NP, pp = k - sub * NP;
    const bool gath = sub < NSUB;
    const int kp = mine ? a.kperm[k] : 0;
    const bool out_cta = g == a.out_cta;
    int bad = -1;
    __syncthreads();
    if (CL > 1) asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    long long tm[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int n = 0; n < a.n_steps; ++n) {
        long long tk = TIMING ? clock64() : 0;
        const float x = (float)q;
        qs[k] = x;                                             // zero beyond n_q
        if (CL > 1 && k == 0) mbar_expect_tx(smem_u32(&rsbar[n & 1]), (uint32_t)(CL * mylen * 4));
        __syncthreads();
        // ---- a2: the thread's item ----------------------------------------------------------------------------
        if (has_item) {
            const float4 *hp = reinterpret_cast<const float4 *>(Hs + I0.x);
            const int ld4 = (I0.y & 0xffff) >> 2;
            const float4 qb = make_float4(qs[I1.x], qs[I1.x + 1], qs[I1.x + 2], qs[I1.x + 3]);   // a class need not start at a multiple of 4
            const float *qa = qs + I0.z;
            float4 c4 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (I1.y >= 0) {
                float *rp = rpart + I1.y;
#pragma unroll 2
                for (int i = 0; i < I0.w; ++i, hp += ld4, rp += I1.z) {
                    const float4 h = *hp; const float qr = qa[i];
                    c4.x = fmaf(h.x, qr, c4.x); c4.y = fmaf(h.y, qr, c4.y); c4.z = fmaf(h.z, qr, c4.z); c4.w = fmaf(h.w, qr, c4.w);
                    *rp = fmaf(h.x, qb.x, fmaf(h.y, qb.y, fmaf(h.z, qb.z, h.w * qb.w)));
                }
            } else {
#pragma unroll 2
                for (int i = 0; i < I0.w; ++i, hp += ld4) {
                    const float4 h = *hp; const float qr = qa[i];
                    c4.x = fmaf(h.x, qr, c4.x); c4.y = fmaf(h.y, qr, c4.y); c4.z = fmaf(h.z, qr, c4.z); c4.w = fmaf(h.w, qr, c4.w);
                }
            }
            *reinterpret_cast<float4 *>(cpart + I1.w) = c4;
        }
        __syncthreads();
        if (TIMING) { const long long t_ = clock64(); tm[0] += t_ - tk; tk = t_; }
        // ---- join (thread k: t_m[k] of every mode of the CTA), a3, a4 ---------------------------------------------------
        float t[MM], vals[8];
#pragma unroll
        for (int m = 0; m < MM; ++m) {
            float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
            if (J[m].x) {
                const float *src = (J[m].x == 2 ? rpart : cpart) + J[m].y;
                const int cnt = J[m].z, st_ = J[m].w;
                int i = 0;
                for (; i + 3 < cnt; i += 4) { a0 += src[i * st_]; a1 += src[(i + 1) * st_]; a2 += src[(i + 2) * st_]; a3 += src[(i + 3) * st_]; }
                for (; i < cnt; ++i) a0 += src[i * st_];
            }
            t[m] = (a0 + a1) + (a2 + a3); vals[m] = x * t[m];
        }
#pragma unroll
        for (int m = MM; m < 8; ++m) vals[m] = 0.f;
        // a1 pickup + a6 write-out ride on the same block sum (slots MM, MM + 1; only the CTA out_cta)
        if (out_cta) { vals[MM] = wk * x; vals[MM + 1] = x * x; }
        if (out_cta) rp_block_sum<MM + 2>(vals, red + (n & 1) * 128);
        else if (MM == 2 || nmodes <= 2) rp_block_sum<2>(vals, red + (n & 1) * 128);
        else rp_block_sum<MM>(vals, red + (n & 1) * 128);
        if (out_cta) {
            if (k == 0) { a.out[n] = vals[MM]; if (bad < 0 && !(isfinite(vals[MM]) && isfinite(vals[MM + 1]))) bad = n; }
            if (a.traj && mine) a.traj[(size_t)n * a.n_q + kp] = q;
        }
        float facc = 0.f;
#pragma unroll
        for (int m = 0; m < MM; ++m) facc = fmaf(sm_[m] * vals[m], t[m], facc);
        if (TIMING) { const long long t_ = clock64(); tm[1] += t_ - tk; tk = t_; }
        // ---- exchange ----------------------------------------------------------------------------------------------
        const unsigned par = (unsigned)n & 1u, epoch = (unsigned)n + 1u;
        unsigned long long *Xp = a.X + (size_t)par * a.NCL * a.NQ2;
        if (CL > 1) {
            if (xk) dsm_st_async1(rs_remote + par * (uint32_t)(CL * SL * 4), bar_remote + par * 8u, facc);
            if (k < mylen) {
                dsm_wait(smem_u32(&rsbar[par]), ((unsigned)n >> 1) & 1u, &s_abort);
                const float *src = rs + (size_t)par * CL * SL + k;
                float fs = 0.f;
                for (int rr = 0; rr < CL; ++rr) fs += src[rr * SL];                 // rank order
                st_tag(Xp + (size_t)cid * a.NQ2 + my0 + k, fs, epoch);
            }
        } else if (xk) {
            st_tag(Xp + (size_t)cid * a.NQ2 + k, facc, epoch);
        }
        if (TIMING) { const long long t_ = clock64(); tm[2] += t_ - tk; tk = t_; }
        if (gath) {                                            // thread (sub, pair): the clusters sub, sub + NSUB, ... of modes 2 pp, 2 pp + 1
            float f0 = 0.f, f1 = 0.f;
            for (int c0 = sub; c0 < a.NCL; c0 += NSUB * RP_GROUND) {
                unsigned long long w0[RP_GROUND], w1[RP_GROUND];
                unsigned pend = 0, spins = 0;
#pragma unroll
                for (int u = 0; u < RP_GROUND; ++u) if (c0 + u * NSUB < a.NCL) pend |= 1u << u;
                const unsigned have = pend;
                while (pend) {
#pragma unroll
                    for (int u = 0; u < RP_GROUND; ++u)
                        if (pend >> u & 1)
                            asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(w0[u]), "=l"(w1[u])
                                         : "l"(Xp + (size_t)(c0 + u * NSUB) * a.NQ2 + 2 * pp) : "memory");
#pragma unroll
                    for (int u = 0; u < RP_GROUND; ++u)
                        if ((pend >> u & 1) && (unsigned)(w0[u] >> 32) == epoch && (unsigned)(w1[u] >> 32) == epoch) pend &= ~(1u << u);
                    if (pend && (++spins & 1023u) == 0 && (s_abort || spins > (1u << 21))) { s_abort = 1; break; }
                }
#pragma unroll
                for (int u = 0; u < RP_GROUND; ++u)
                    if (have >> u & 1) { f0 += __uint_as_float((unsigned)w0[u]); f1 += __uint_as_float((unsigned)w1[u]); }
            }
            *reinterpret_cast<float2 *>(part2 + (size_t)sub * RP_THREADS + 2 * pp) = make_float2(f0, f1);
        }
        __syncthreads();
        if (TIMING) { const long long t_ = clock64(); tm[3] += t_ - tk; tk = t_; }
        float f = 0.f;
        if (mine) for (int xx = 0; xx < NSUB; ++xx) f += part2[xx * RP_THREADS + k];
        // ---- a5 --------------------------------------------------------------------------------------------------------
        const double fd = (double)f;
        if (n == 0 && a.auto_start) v = (r != 0.0) ? ast * q + a.half_T2 * fd : 0.0;
        const double fe = a.fext ? (double)a.fext[n] * gn : 0.0;
        v = kv * v - kq * q + r * (fe - fd);
        q += v;
        // qs, cpart, rpart, part2 are rewritten only after the next step's first barrier / item barrier
    }
    if (out_cta && k == 0) a.first_bad[0] = bad;
    if (k == 0 && s_abort) *a.timeout_flag = 1;
    if (TIMING && k == 0) for (int x = 0; x < 8; ++x) a.timing[(size_t)g * 8 + x] = tm[x];
    if (CL > 1) {   // no CTA of the cluster leaves while a peer may still store into its shared memory
        __syncthreads();
        asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
}

}  // namespace modal_dev
