// vk_bptt.cuh -- reverse pass (backpropagation through time) of the von Karman recurrence: SURVEY.md 8(f) row 3,
// PAPER.md:281-285 ("gradients ... by backpropagation through the time integrator"; the paper uses autodiff, this is the same
// adjoint as hand-written kernels).  Oracle: oracle.bptt_vk.  DESIGN.md 7.6.
//
// Forward (Eq. 19/20):  out_n = w . q^n,   q^{n+1} = c1 q^n + c2 q^{n-1} - c3 f(q^n),
//   f_k = sum_m s_m G_m t_mk,  t_m = H^m q,  G_m = q . t_m   (Eq. 9, C eliminated by PAPER.md:283)
// Adjoint a^n = dL/dq^n, a^N = a^{N+1} = 0, gout_n = dL/d out_n, mu = c3 a^{n+1}, H^m symmetric:
//   a^n = w gout_n + c1 a^{n+1} + c2 a^{n+2} - sum_m s_m [ 2 (t_m . mu) t_m + G_m H^m mu ]
//   dL/dc1 += a^{n+1} q^n;  dL/dc2 += a^{n+1} q^{n-1};  dL/dc3 -= a^{n+1} f(q^n);  dL/dw += gout_n q^n;  dL/ds_m -= (t_m . mu) G_m
//   dL/dH^m_kr = - sum_{b,n} [ s_m (t_m . mu) q_k + s_m G_m mu_k ] q_r        (vk_gradH_kernel, from the stored mu^n and scalars)
//
// vk_bptt_kernel: a team of G CTAs per sample, the in-plane modes m split over the team; per reverse step each CTA reads the rows
// of its H^m ONCE for both contractions (t_m = H^m q and u_m = H^m mu; H^m resident in shared memory when the CTA's modes fit), the partial Jacobian product
// and the partial force are exchanged as tagged 64-bit words {fp32, epoch} through L2 (st_tag / ld_tag of vk_flow.cuh, every wait
// bounded) and summed in team order, so every CTA of the team carries a bit-identical fp64 replica of the adjoint state.
// Contractions in fp32 (as the forward path), adjoint state and gradient accumulators in fp64.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_flow.cuh"

namespace modal_dev {

constexpr int BP_THREADS_MAX = 512;     // one thread per transverse mode: n_q <= 512; the kernel always runs 512 threads (16 warps share the rows)
constexpr int BP_G_MAX = 32;             // CTAs of a team (also bounded by 8 x (512 / row stride): eight sources per gathering thread)

struct BpttArgs {
    int n_q, n_phi, batch, n_steps, G, cb_q, cb_phi;        // cb_*: coefficient row stride per sample (0: one row for all)
    int ld, NJ;                                             // row stride of H (n_q rounded up to 4), row groups of the contraction pass
    const float *H;                                         // dense [n_phi][n_q][ld], plan order, rows zero-padded
    const double *c1, *c2, *c3; const float *s, *w;         // plan order, masked modes zero
    const double *traj;                                     // [batch][n_steps][n_q]  q^n of the forward run
    const double *qm1;                                      // [batch][n_q]
    const float *gout;                                      // [batch][n_steps]
    double *g_q0, *g_qm1, *g_c1, *g_c2, *g_c3, *g_w;        // [batch][n_q]
    double *g_s;                                            // [batch][n_phi]
    float *mu_traj;                                         // optional [batch][n_steps][n_q]: mu^n = c3 a^{n+1}   (for dL/dH)
    float *dsc, *esc;                                       // optional [batch][n_steps][n_phi]: s_m (t_m . mu), s_m G_m
    unsigned long long *scratch;                            // [2][batch][G][n_q][2] tagged words
    int *timeout_flag;
};

// sums of a and b over the block, in a fixed order; every thread gets both.  red: 2 * 16 floats.  Two barriers.
__device__ __forceinline__ void bp_block_sum2(float a, float b, float *red, int nwarps, float &A, float &B)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) { a += __shfl_xor_sync(FLOW_FULL, a, m); b += __shfl_xor_sync(FLOW_FULL, b, m); }
    if (lane == 0) { red[warp] = a; red[16 + warp] = b; }
    __syncthreads();
    // lane y reads the sums of warp y, a 16-lane butterfly joins them (a loop of dependent shared-memory loads cost ~500 cycles here)
    const int y = lane & 15;
    A = y < nwarps ? red[y] : 0.f; B = y < nwarps ? red[16 + y] : 0.f;
#pragma unroll
    for (int m = 8; m >= 1; m >>= 1) { A += __shfl_xor_sync(FLOW_FULL, A, m); B += __shfl_xor_sync(FLOW_FULL, B, m); }
    __syncthreads();
}

template <bool RESIDENT>
__global__ void __launch_bounds__(BP_THREADS_MAX) vk_bptt_kernel(const BpttArgs a)
{
    __shared__ float2 qm[BP_THREADS_MAX];                    // (q^n_r, mu_r)
    __shared__ __align__(16) float part[2 * 2048];           // partial t and u vectors of the NJ row groups
    __shared__ float red[32];
    __shared__ volatile int s_abort;
    __shared__ double gsacc[256];                            // dL/ds_m of the CTA's modes (global memory beyond 256 modes per CTA)
    extern __shared__ __align__(16) float Hs[];              // resident: [modes of this CTA][n_q][ld]
    const int k = threadIdx.x, nwarps = blockDim.x >> 5;
    const int ld = a.ld, NQ4 = ld >> 2, NJ = a.NJ, RJ = (a.n_q + NJ - 1) / NJ;
    const int jg = k / NQ4, cq4 = k - jg * NQ4;
    const bool pass_on = jg < NJ;
    const int r0 = min(a.n_q, jg * RJ), r1 = min(a.n_q, r0 + RJ);
    const int bl = blockIdx.x / a.G, g = blockIdx.x - bl * a.G;
    const int m0 = (int)((long long)a.n_phi * g / a.G), m1 = (int)((long long)a.n_phi * (g + 1) / a.G);
    const bool mine = k < a.n_q;
    const size_t cq = (size_t)bl * a.cb_q, cp = (size_t)bl * a.cb_phi;
    double c1 = 0.0, c2 = 0.0, c3 = 0.0; float wk = 0.f;
    if (mine) { c1 = a.c1[cq + k]; c2 = a.c2[cq + k]; c3 = a.c3[cq + k]; wk = a.w[cq + k]; }
    double a1 = 0.0, a2 = 0.0;                               // a^{n+1}, a^{n+2}
    double gc1 = 0.0, gc2 = 0.0, gc3 = 0.0, gw = 0.0;
    if (k == 0) s_abort = 0;
    if (k < 256) gsacc[k] = 0.0;
    const bool gs_local = m1 - m0 <= 256;
    if (RESIDENT) {
        const float *src = a.H + (size_t)m0 * a.n_q * ld;
        const size_t cnt = (size_t)(m1 - m0) * a.n_q * ld;
        for (size_t i = k; i < cnt; i += blockDim.x) Hs[i] = __ldg(src + i);
    }
    const float *s = a.s + cp;
    const double *traj = a.traj + (size_t)bl * a.n_steps * a.n_q;
    const float *gout = a.gout + (size_t)bl * a.n_steps;
    // q^n and q^{n-1} travel in registers; the one new value per step (q^{n-2}) is loaded at the top of the step, a step ahead of its use
    const double *tk_ = traj + k;
    const double qm1k = mine ? a.qm1[(size_t)bl * a.n_q + k] : 0.0;
    double qn = mine ? tk_[(size_t)(a.n_steps - 1) * a.n_q] : 0.0;
    double qp = !mine ? 0.0 : a.n_steps >= 2 ? tk_[(size_t)(a.n_steps - 2) * a.n_q] : qm1k;
    float go_next = gout[a.n_steps - 1];
    for (int n = a.n_steps - 1; n >= 0; --n) {
        double qpp = 0.0;
        if (mine) qpp = n >= 2 ? tk_[(size_t)(n - 2) * a.n_q] : (n == 1 ? qm1k : 0.0);
        const float go_f = go_next;
        if (n > 0) go_next = gout[n - 1];
        const double mu = c3 * a1;
        const float x = (float)qn, y = (float)mu;
        qm[k] = make_float2(x, y);
        if (g == 0 && mine && a.mu_traj) a.mu_traj[((size_t)bl * a.n_steps + n) * a.n_q + k] = y;
        __syncthreads();
        float jacc = 0.f, facc = 0.f;
        for (int m = m0; m < m1; ++m) {
            const float *Hm = RESIDENT ? Hs + (size_t)(m - m0) * a.n_q * ld : a.H + (size_t)m * a.n_q * ld;
            // both contractions from ONE read of H^m: thread (jg, cq4) multiplies rows r0..r1 of its four columns (16-byte loads,
            // consecutive threads consecutive addresses); q_r and mu_r are broadcast reads.  H^m is symmetric, so the column sums
            // sum_r H[r][k] x_r are (H^m x)_k.  No shuffles; the NJ partial vectors are joined through shared memory.
            float4 t4 = make_float4(0.f, 0.f, 0.f, 0.f), u4 = t4;
            if (pass_on) {
                const float *hp = Hm + (size_t)r0 * ld + 4 * cq4;
#pragma unroll 4
                for (int r = r0; r < r1; ++r, hp += ld) {
                    const float4 h = RESIDENT ? *reinterpret_cast<const float4 *>(hp) : __ldg(reinterpret_cast<const float4 *>(hp));
                    const float2 v = qm[r];
                    t4.x = fmaf(h.x, v.x, t4.x); t4.y = fmaf(h.y, v.x, t4.y); t4.z = fmaf(h.z, v.x, t4.z); t4.w = fmaf(h.w, v.x, t4.w);
                    u4.x = fmaf(h.x, v.y, u4.x); u4.y = fmaf(h.y, v.y, u4.y); u4.z = fmaf(h.z, v.y, u4.z); u4.w = fmaf(h.w, v.y, u4.w);
                }
                *reinterpret_cast<float4 *>(part + (size_t)jg * ld + 4 * cq4) = t4;
                *reinterpret_cast<float4 *>(part + 2048 + (size_t)jg * ld + 4 * cq4) = u4;
            }
            __syncthreads();
            float t = 0.f, u = 0.f;
            if (mine)
                for (int jj = 0; jj < NJ; ++jj) { t += part[jj * ld + k]; u += part[2048 + jj * ld + k]; }      // group order (deterministic)
            float Gm, dm;
            bp_block_sum2(x * t, y * t, red, nwarps, Gm, dm);             // G_m = q . t_m,  d_m = mu . t_m
            const float sm = s[m];
            jacc = fmaf(sm * dm, 2.f * t, fmaf(sm * Gm, u, jacc));
            facc = fmaf(sm * Gm, t, facc);
            if (k == 0) {
                if (gs_local) gsacc[m - m0] -= (double)dm * (double)Gm;          // this CTA owns mode m of this sample
                else a.g_s[(size_t)bl * a.n_phi + m] -= (double)dm * (double)Gm;
                if (a.dsc) {
                    a.dsc[((size_t)bl * a.n_steps + n) * a.n_phi + m] = sm * dm;
                    a.esc[((size_t)bl * a.n_steps + n) * a.n_phi + m] = sm * Gm;
                }
            }
        }
        float J = jacc, f = facc;
        if (a.G > 1) {
            const unsigned epoch = (unsigned)(a.n_steps - n);
            unsigned long long *base = a.scratch + ((((size_t)(n & 1) * a.batch + bl) * a.G) * a.n_q) * 2;
            if (mine) {
                st_tag(base + ((size_t)g * a.n_q + k) * 2, jacc, epoch);
                st_tag(base + ((size_t)g * a.n_q + k) * 2 + 1, facc, epoch);
            }
            // gather: thread (sub, kk) takes the sources sub, sub + NSUB, ... (at most eight, all in flight together) of mode kk; the
            // sub-group partials are joined through shared memory in sub order: every CTA of the team adds the same numbers in the same order
            const int NSUB = min(BP_THREADS_MAX / ld, 8);
            const int sub = k / ld, kk = k - sub * ld;
            if (sub < NSUB && kk < a.n_q) {
                float2 v[8];
                unsigned pend = 0, spins = 0;
#pragma unroll
                for (int u = 0; u < 8; ++u) if (sub + u * NSUB < a.G) pend |= 1u << u;
                const unsigned have = pend;
                while (pend) {
                    unsigned long long w0[8], w1[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (pend >> u & 1)
                            asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(w0[u]), "=l"(w1[u])
                                         : "l"(base + ((size_t)(sub + u * NSUB) * a.n_q + kk) * 2) : "memory");
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if ((pend >> u & 1) && (unsigned)(w0[u] >> 32) == epoch && (unsigned)(w1[u] >> 32) == epoch) {
                            v[u] = make_float2(__uint_as_float((unsigned)w0[u]), __uint_as_float((unsigned)w1[u]));
                            pend &= ~(1u << u);
                        }
                    if (pend && (++spins & 1023u) == 0 && (s_abort || spins > (1u << 21))) { s_abort = 1; break; }
                }
                float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                for (int u = 0; u < 8; ++u) if (have >> u & 1) { acc.x += v[u].x; acc.y += v[u].y; }
                *reinterpret_cast<float2 *>(part + 2 * (sub * ld + kk)) = acc;
            }
            __syncthreads();
            if (mine) {
                J = 0.f; f = 0.f;
                for (int x = 0; x < NSUB; ++x) { const float2 p2 = *reinterpret_cast<const float2 *>(part + 2 * (x * ld + k)); J += p2.x; f += p2.y; }
            }
        }
        const double go = (double)go_f;
        gc1 = fma(a1, qn, gc1); gc2 = fma(a1, qp, gc2); gc3 = fma(-a1, (double)f, gc3); gw = fma(go, qn, gw);
        const double a0 = fma((double)wk, go, fma(c1, a1, fma(c2, a2, -(double)J)));
        a2 = a1; a1 = a0;
        qn = qp; qp = qpp;
        __syncthreads();
    }
    if (g == 0 && mine) {
        const size_t o = (size_t)bl * a.n_q + k;
        a.g_q0[o] = a1; a.g_qm1[o] = c2 * a2;
        a.g_c1[o] = gc1; a.g_c2[o] = gc2; a.g_c3[o] = gc3; a.g_w[o] = gw;
    }
    if (gs_local && k < m1 - m0) a.g_s[(size_t)bl * a.n_phi + m0 + k] = gsacc[k];
    if (k == 0 && s_abort) *a.timeout_flag = 1;
}

// dL/dH^m_kr = - sum_b sum_n (D[b][n][m] q^n_k + E[b][n][m] mu^n_k) q^n_r :  block = (mode m, 16 rows k), thread = column r;
// samples and steps in order (deterministic, no atomics).
__global__ void __launch_bounds__(BP_THREADS_MAX) vk_gradH_kernel(int n_q, int n_phi, int batch, int n_steps, const double *traj,
                                                                  const float *mu_traj, const float *dsc, const float *esc, double *gH)
{
    __shared__ float xk[16];
    const int m = blockIdx.x, k0 = blockIdx.y * 16, r = threadIdx.x;
    double acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = 0.0;
    for (int b = 0; b < batch; ++b)
        for (int n = 0; n < n_steps; ++n) {
            const size_t o = (size_t)b * n_steps + n;
            if (r < 16) {
                const int kk = k0 + r;
                xk[r] = kk < n_q ? dsc[o * n_phi + m] * (float)traj[o * n_q + kk] + esc[o * n_phi + m] * mu_traj[o * n_q + kk] : 0.f;
            }
            __syncthreads();
            const float qr = r < n_q ? (float)traj[o * n_q + r] : 0.f;
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[i] -= (double)(xk[i] * qr);
            __syncthreads();
        }
    if (r < n_q)
        for (int i = 0; i < 16; ++i)
            if (k0 + i < n_q) gH[((size_t)m * n_q + k0 + i) * n_q + r] = acc[i];
}

}  // namespace modal_dev

namespace modal_dev {

// ---- reverse pass of the tension-modulated / linear recurrence (Kirchhoff-Carrier string, Berger plate): one warp per sample --------
//   f_mu = c lam_mu q_mu S,  S = sum lam q^2  (Eq. 8, reading R2);  J symmetric:
//   J^T mu = c [ S lam mu + 2 (sum lam q mu) lam q ];   dL/dc -= (sum lam q mu) S;   the rest as vk_bptt_kernel.  Oracle: oracle.bptt_tension.
// O(N) work per step: the adjoint state and the gradient accumulators of a sample live in the warp's slice of shared memory (fp64).
constexpr int TB_WARPS = 4;

struct TensionBpttArgs {
    int n_q, batch, n_steps, cb_q;                         // cb_q: coefficient row stride per sample (0: one row for all)
    const double *c1, *c2, *c3; const float *w, *lam, *c;  // [cb][n_q] ...; c [cb]
    const double *traj, *qm1; const float *gout;
    double *g_q0, *g_qm1, *g_c1, *g_c2, *g_c3, *g_w, *g_c; // [batch][n_q]; g_c [batch]
};

__host__ __device__ inline size_t tension_bptt_smem(int n_q) { return (size_t)TB_WARPS * n_q * 6 * sizeof(double); }

__global__ void __launch_bounds__(TB_WARPS * 32) tension_bptt_kernel(const TensionBpttArgs a)
{
    extern __shared__ __align__(16) double tb_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.x * TB_WARPS + warp;
    if (b >= a.batch) return;
    const int nq = a.n_q;
    double *A1 = tb_smem + (size_t)warp * nq * 6, *A2 = A1 + nq, *G1 = A2 + nq, *G2 = G1 + nq, *G3 = G2 + nq, *GW = G3 + nq;
    for (int k = lane; k < nq; k += 32) { A1[k] = 0.0; A2[k] = 0.0; G1[k] = 0.0; G2[k] = 0.0; G3[k] = 0.0; GW[k] = 0.0; }
    __syncwarp();
    const size_t co = (size_t)b * a.cb_q;
    const double *c1 = a.c1 + co, *c2 = a.c2 + co, *c3 = a.c3 + co;
    const float *w = a.w + co, *lam = a.lam + co;
    const double cn = (double)a.c[a.cb_q ? b : 0];
    const double *traj = a.traj + (size_t)b * a.n_steps * nq, *qm1 = a.qm1 + (size_t)b * nq;
    double gcn = 0.0;
    for (int n = a.n_steps - 1; n >= 0; --n) {
        const double *qn = traj + (size_t)n * nq;
        const double *qp = n > 0 ? traj + (size_t)(n - 1) * nq : qm1;
        double S = 0.0, D = 0.0;
        for (int k = lane; k < nq; k += 32) {
            const double q = qn[k], lq = (double)lam[k] * q;
            S = fma(lq, q, S); D = fma(lq, c3[k] * A1[k], D);
        }
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) { S += __shfl_xor_sync(FLOW_FULL, S, m); D += __shfl_xor_sync(FLOW_FULL, D, m); }
        const double go = (double)a.gout[(size_t)b * a.n_steps + n];
        for (int k = lane; k < nq; k += 32) {
            const double q = qn[k], l = (double)lam[k], a1 = A1[k], mu = c3[k] * a1;
            const double f = cn * l * q * S;
            const double JT = cn * (S * l * mu + 2.0 * D * l * q);
            G1[k] = fma(a1, q, G1[k]); G2[k] = fma(a1, qp[k], G2[k]); G3[k] = fma(-a1, f, G3[k]); GW[k] = fma(go, q, GW[k]);
            const double a0 = fma((double)w[k], go, fma(c1[k], a1, fma(c2[k], A2[k], -JT)));
            A2[k] = a1; A1[k] = a0;
        }
        gcn -= D * S;
        __syncwarp();
    }
    for (int k = lane; k < nq; k += 32) {
        const size_t o = (size_t)b * nq + k;
        a.g_q0[o] = A1[k]; a.g_qm1[o] = c2[k] * A2[k]; a.g_c1[o] = G1[k]; a.g_c2[o] = G2[k]; a.g_c3[o] = G3[k]; a.g_w[o] = GW[k];
    }
    if (lane == 0) a.g_c[b] = gcn;
}

}  // namespace modal_dev
