// kernels.cuh -- hand-written sm_100a kernels of the modal hot path.
//
//   tension_kernel : MODAL_LINEAR / MODAL_TENSION, one warp per sample, state in registers
//                    (Eq. 8 + PAPER.md:153-167 Eq. 19-23).
// The MODAL_VK kernels live in vk_flow.cuh (FP32 pipe, small batch) and vk_mma.cuh (tcgen05, wide batch).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace modal_dev {

constexpr unsigned FULL = 0xffffffffu;

// ----------------------------------------------------------------------------------------
// Delta form of the two-step update: with v^n = q^n - q^{n-1}
//   v^{n+1} = kv v^n - kq q^n + r (fext - fnl),   q^{n+1} = q^n + v^{n+1}
// SV : kv = (1-gT)/(1+gT), kq = r w^2, r = T^2/(1+gT)   (== Eq. 20-23: g = 1+kv-kq, p = -kv)
// FTM: kv = a2, kq = 1+a1+a2, r = b1                    (== Eq. 16-19 with -a1, -a2)
// State and coefficients are fp64; the vK force is evaluated in fp32 (tension kernel: per-lane sums in
// fp64, the cross-lane sums S and pickup in fp32).
// ----------------------------------------------------------------------------------------

struct TensionArgs {
    int batch, n_steps, n_modes_pad;     // n_modes_pad = 32 * MPL
    int coeff_stride;                    // 0 (shared coefficients) or n_modes_pad
    const double *kv, *kq, *r, *astart;  // [cb][pad]
    const float *lambda, *w;             // [cb][pad]
    const float *c;                      // [cb]   tau / rho_m (0 for MODAL_LINEAR)
    const double *q0, *v0;               // [batch][pad]
    int auto_start; double half_T2;      // v0 = astart q0 + half_T2 fnl(q0) on active modes
    const float *fext; const double *gain;  // optional [batch][n_steps], [batch][pad]
    float *out; double *traj; int n_q;   // out [batch][n_steps]; traj optional [batch][n_steps][n_q]
    int *first_bad;                      // [batch]
};

template <int MPL>
__global__ void __launch_bounds__(128) tension_kernel(const TensionArgs a)
{
    const int lane = threadIdx.x & 31;
    const int b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (b >= a.batch) return;
    const size_t co = (size_t)(a.coeff_stride ? b : 0) * a.n_modes_pad;
    const size_t so = (size_t)b * a.n_modes_pad;
    // rl = r * lambda: the force term r f_mu = (r lambda_mu)(c S) q_mu is folded into the fp64 update, so the
    // step has no per-mode conversion between fp32 and fp64 (only S and the pickup cross the lanes, in fp32)
    double q[MPL], v[MPL], kv[MPL], kq[MPL], rl[MPL], rg[MPL], lam[MPL], w[MPL];
#pragma unroll
    for (int j = 0; j < MPL; ++j) {
        const int k = lane + 32 * j;
        q[j] = a.q0[so + k]; v[j] = a.v0[so + k];
        kv[j] = a.kv[co + k]; kq[j] = a.kq[co + k];
        lam[j] = a.lambda[co + k]; w[j] = a.w[co + k];
        const double r = a.r[co + k];
        rl[j] = r * lam[j];
        rg[j] = a.fext ? r * a.gain[so + k] : 0.0;
    }
    const float c = a.c[a.coeff_stride ? b : 0];
    float oreg = 0.f;
    int bad = -1;
    float *out = a.out + (size_t)b * a.n_steps;
    for (int n = 0; n < a.n_steps; ++n) {
        // per-lane partial sums in fp64 straight from the state (no per-mode conversion; two chains each),
        // rounded to fp32 once for the shuffle reduction
        double od = 0.0, Sd = 0.0, od1 = 0.0, Sd1 = 0.0;
#pragma unroll
        for (int j = 0; j < MPL; ++j) {
            if (j & 1) { od1 = fma(w[j], q[j], od1); Sd1 = fma(lam[j] * q[j], q[j], Sd1); }
            else       { od = fma(w[j], q[j], od);   Sd = fma(lam[j] * q[j], q[j], Sd); }
        }
        float o = (float)(od + od1), S = (float)(Sd + Sd1);
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
            o += __shfl_xor_sync(FULL, o, m);
            S += __shfl_xor_sync(FULL, S, m);
        }
        if (bad < 0 && !(isfinite(o) && isfinite(S))) bad = n;
        if ((n & 31) == lane) oreg = o;
        if ((n & 31) == 31) out[n - 31 + lane] = oreg;
        if (a.traj) {
#pragma unroll
            for (int j = 0; j < MPL; ++j) {
                const int k = lane + 32 * j;
                if (k < a.n_q) a.traj[((size_t)b * a.n_steps + n) * a.n_q + k] = q[j];
            }
        }
        const double cS = (double)(c * S);
        const double fe = a.fext ? (double)a.fext[(size_t)b * a.n_steps + n] : 0.0;
        if (n == 0 && a.auto_start) {
#pragma unroll
            for (int j = 0; j < MPL; ++j)
                v[j] = (a.r[co + lane + 32 * j] != 0.0)
                           ? a.astart[co + lane + 32 * j] * q[j] + a.half_T2 * (cS * lam[j] * q[j]) : 0.0;
        }
#pragma unroll
        for (int j = 0; j < MPL; ++j) {
            v[j] = fma(-fma(rl[j], cS, kq[j]), q[j], fma(kv[j], v[j], fe * rg[j]));   // only the first factor waits for S
            q[j] += v[j];
        }
    }
    const int rem = a.n_steps & 31;
    if (rem && lane < rem) out[a.n_steps - rem + lane] = oreg;
    if (lane == 0) a.first_bad[b] = bad;
}

}  // namespace modal_dev
