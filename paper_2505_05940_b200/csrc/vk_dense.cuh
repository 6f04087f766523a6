// vk_dense.cuh -- von Karman time loop for MID-SIZE systems at small batch (the paper's 50- and 100-mode benchmark points,
// PAPER.md:192-203; BASELINE.json config 2): a team of G <= 32 CTAs per sample with ONE cross-CTA hop per step.
//
// vk_flow_kernel needs two L2 hops per step (partial forces -> owners, new state -> everybody) and five CTA-wide phases; at
// 100 + 50 modes that is 8.7 k cycles per step of which 1.7 k are the contraction (profiles/r2_batch1_latency.md).  Here every CTA
// of the team keeps the WHOLE fp64 state (thread k <-> mode k, bit-identical replicas), the in-plane modes are split over the team,
// and the only exchange is the all-gather of the partial forces (tagged 64-bit words {fp32, epoch} through L2, double-buffered by
// step parity, gathered by sub-groups of threads with all loads in flight, summed in a fixed order).  H^m of the CTA's modes is
// dense fp32 in shared memory (internal mode order, rows padded to 16 bytes); thread (row group, column quad) reads 16 bytes per
// row and the row-group partials are joined through shared memory -- no shuffles.  H^m symmetric: column sums are (H^m q)_k.
//   t_m = H^m q;  G_m = q . t_m;  eta_m = s_m G_m;  f = sum_m eta_m t_m          (a2-a4; Eq. 9-11, C eliminated :283)
//   v <- kv v - kq q + r (fext - f),  q <- q + v                                  (a5; Eq. 19/20, delta form)
//   out[b][n] = w . q^n  by the CTA `out_cta` of the team                         (a1, a6)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_flow.cuh"

namespace modal_dev {

constexpr int DN_THREADS = 512;         // thread k <-> mode k: n_q <= 512
constexpr int DN_G_MAX = 32;

struct DenseArgs {
    int n_q, n_phi, NQP, batch, n_steps, G, ld, NJ, out_cta;
    int coeff_stride_q, coeff_stride_phi;
    const float *H;                      // dense [n_phi][n_q][ld], internal mode order, rows zero-padded
    const double *kv, *kq, *r, *astart;
    const float *s, *w;
    const double *q0, *v0;
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; const int *kperm; int *first_bad;
    unsigned long long *scratch;         // [2][samples of the launch][G][n_q] tagged words
    int *timeout_flag;
};

// sum of a over the block, fixed order; every thread gets the same bits.  red: 16 floats.  Two barriers.  The 16 warp sums are joined
// by a 16-lane butterfly (lane y reads the sum of warp y): 16 dependent shared-memory loads per thread measured 640 cycles, this ~150.
__device__ __forceinline__ float dn_block_sum(float a, float *red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) a += __shfl_xor_sync(FLOW_FULL, a, m);
    if (lane == 0) red[warp] = a;
    __syncthreads();
    float A = red[lane & 15];
#pragma unroll
    for (int m = 8; m >= 1; m >>= 1) A += __shfl_xor_sync(FLOW_FULL, A, m);
    __syncthreads();
    return A;
}
// two values at once (the pickup and the norm of the state).  red: 32 floats.
__device__ __forceinline__ void dn_block_sum2(float &a, float &b, float *red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) { a += __shfl_xor_sync(FLOW_FULL, a, m); b += __shfl_xor_sync(FLOW_FULL, b, m); }
    if (lane == 0) { red[warp] = a; red[16 + warp] = b; }
    __syncthreads();
    float A = red[lane & 15], B = red[16 + (lane & 15)];
#pragma unroll
    for (int m = 8; m >= 1; m >>= 1) { A += __shfl_xor_sync(FLOW_FULL, A, m); B += __shfl_xor_sync(FLOW_FULL, B, m); }
    __syncthreads();
    a = A; b = B;
}

__global__ void __launch_bounds__(DN_THREADS) vk_dense_kernel(const DenseArgs a)
{
    __shared__ float qs[DN_THREADS];
    __shared__ __align__(16) float part[2048];               // partial t vectors of the NJ row groups; partial forces of the gather sub-groups
    __shared__ float red[32];
    __shared__ volatile int s_abort;
    extern __shared__ __align__(16) float Hs[];              // [modes of this CTA][n_q][ld]
    const int k = threadIdx.x;
    const int ld = a.ld, NQ4 = ld >> 2, NJ = a.NJ, RJ = (a.n_q + NJ - 1) / NJ;
    const int jg = k / NQ4, cq4 = k - jg * NQ4;
    const bool pass_on = jg < NJ;
    const int r0 = min(a.n_q, jg * RJ), r1 = min(a.n_q, r0 + RJ);
    const int bl = blockIdx.x / a.G, g = blockIdx.x - bl * a.G;
    const int m0 = (int)((long long)a.n_phi * g / a.G), m1 = (int)((long long)a.n_phi * (g + 1) / a.G);
    const bool mine = k < a.n_q;
    const size_t co = (size_t)(a.coeff_stride_q ? bl : 0) * a.NQP + k;
    double q = 0.0, v = 0.0, kv = 0.0, kq = 0.0, r = 0.0, ast = 0.0, gn = 0.0; float wk = 0.f;
    if (mine) {
        q = a.q0[(size_t)bl * a.NQP + k]; v = a.v0[(size_t)bl * a.NQP + k];
        kv = a.kv[co]; kq = a.kq[co]; r = a.r[co]; ast = a.astart[co]; wk = a.w[co];
        if (a.fext) gn = a.gain[(size_t)bl * a.NQP + k];
    }
    if (k == 0) s_abort = 0;
    {
        const float *src = a.H + (size_t)m0 * a.n_q * ld;
        const size_t cnt = (size_t)(m1 - m0) * a.n_q * ld;
        for (size_t i = k; i < cnt; i += blockDim.x) Hs[i] = __ldg(src + i);
    }
    const float *s = a.s + (size_t)(a.coeff_stride_phi ? bl : 0) * a.n_phi;
    const int kp = mine ? a.kperm[k] : 0;
    const bool out_cta = g == a.out_cta;
    const int NSUB = min(DN_THREADS / ld, 8);
    const int sub = k / ld, kk = k - sub * ld;
    int bad = -1;
    float *out = a.out + (size_t)bl * a.n_steps;
    __syncthreads();
    for (int n = 0; n < a.n_steps; ++n) {
        const float x = (float)q;
        qs[k] = x;                                           // zero beyond n_q
        __syncthreads();
        if (out_cta) {                                       // a1 pickup + a6 write-out (the CTA with the fewest modes)
            float o = wk * x, nr = x * x;
            dn_block_sum2(o, nr, red);
            if (k == 0) { out[n] = o; if (bad < 0 && !(isfinite(o) && isfinite(nr))) bad = n; }
            if (a.traj && mine) a.traj[((size_t)bl * a.n_steps + n) * a.n_q + kp] = q;
        }
        float facc = 0.f;
        for (int m = m0; m < m1; ++m) {
            const float *Hm = Hs + (size_t)(m - m0) * a.n_q * ld;
            float4 t4 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (pass_on) {
                const float *hp = Hm + (size_t)r0 * ld + 4 * cq4;
#pragma unroll 4
                for (int rr = r0; rr < r1; ++rr, hp += ld) {
                    const float4 h = *reinterpret_cast<const float4 *>(hp);
                    const float qr = qs[rr];
                    t4.x = fmaf(h.x, qr, t4.x); t4.y = fmaf(h.y, qr, t4.y); t4.z = fmaf(h.z, qr, t4.z); t4.w = fmaf(h.w, qr, t4.w);
                }
                *reinterpret_cast<float4 *>(part + (size_t)jg * ld + 4 * cq4) = t4;
            }
            __syncthreads();
            float t = 0.f;
            if (mine)
                for (int jj = 0; jj < NJ; ++jj) t += part[jj * ld + k];          // group order (deterministic)
            const float Gm = dn_block_sum(x * t, red);                           // its second barrier also protects part
            facc = fmaf(s[m] * Gm, t, facc);
        }
        float f = facc;
        if (a.G > 1) {
            const unsigned epoch = (unsigned)n + 1u;
            unsigned long long *base = a.scratch + (((size_t)(n & 1) * (gridDim.x / a.G) + bl) * a.G) * a.n_q;
            if (mine) st_tag(base + (size_t)g * a.n_q + k, facc, epoch);
            if (sub < NSUB && kk < a.n_q) {                  // thread (sub, kk): the sources sub, sub + NSUB, ... of mode kk, all in flight
                float vv[8];
                unsigned pend = 0, spins = 0;
#pragma unroll
                for (int u = 0; u < 8; ++u) if (sub + u * NSUB < a.G) pend |= 1u << u;
                const unsigned have = pend;
                while (pend) {
                    unsigned long long w0[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (pend >> u & 1)
                            asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(w0[u]) : "l"(base + (size_t)(sub + u * NSUB) * a.n_q + kk) : "memory");
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if ((pend >> u & 1) && (unsigned)(w0[u] >> 32) == epoch) { vv[u] = __uint_as_float((unsigned)w0[u]); pend &= ~(1u << u); }
                    if (pend && (++spins & 1023u) == 0 && (s_abort || spins > (1u << 21))) { s_abort = 1; break; }
                }
                float acc = 0.f;
#pragma unroll
                for (int u = 0; u < 8; ++u) if (have >> u & 1) acc += vv[u];
                part[sub * ld + kk] = acc;
            }
            __syncthreads();
            f = 0.f;
            if (mine) for (int xx = 0; xx < NSUB; ++xx) f += part[xx * ld + k];
        }
        const double fd = (double)f;
        if (n == 0 && a.auto_start) v = (r != 0.0) ? ast * q + a.half_T2 * fd : 0.0;
        const double fe = a.fext ? (double)a.fext[(size_t)bl * a.n_steps + n] * gn : 0.0;
        v = kv * v - kq * q + r * (fe - fd);
        q += v;
        __syncthreads();                                     // qs and part are rewritten in the next step
    }
    if (out_cta && k == 0) a.first_bad[bl] = bad;
    if (k == 0 && s_abort) *a.timeout_flag = 1;
}

}  // namespace modal_dev
