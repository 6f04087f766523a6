// vk_small.cuh -- von Karman time loop of SMALL systems (N_q <= 32, N_phi <= 32, N_phi N_q^2 <= 8192: the paper's 10-mode benchmark
// point, BASELINE.json config 0): one WARP per sample, no CTA barrier, no cross-CTA exchange.
//
// At these sizes a step is a few hundred dependent cycles of arithmetic; the phase structure of vk_flow_kernel (five CTA-wide
// barriers, 16 warps) costs 4 k cycles per step however small the system (profiles/r2_batch1_latency.md).  Here the dense fp32 H
// (internal mode order, as unpacked from the flow tiles) sits in shared memory once per CTA and each warp advances its own sample:
//   t[n][k] = sum_r H^n[k][r] q_r        lanes share the (n, k) pairs; q_r are broadcast reads from shared memory        (a2)
//   G_n = sum_k q_k t[n][k], eta_n = s_n G_n   lane n                                                                    (a3, a4)
//   f_k = sum_n eta_n t[n][k]            lane k; fp64 delta-form update v <- kv v - kq q + r (fext - f), q <- q + v     (a5)
//   out[b][n] = sum_k w_k q_k^n          warp shuffle reduction, written in 128-byte rows                                (a1, a6)
// (Eq. 9-11 with C eliminated; Eq. 19/20.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "vk_flow.cuh"   // FLOW_FULL

namespace modal_dev {

constexpr int SM_WARPS = 4;             // samples per CTA
constexpr int SM_TS = 33;               // row stride of t[n][.] (odd: lane n reads row n without bank conflicts)

struct SmallArgs {
    const float *Hd;            // dense [n_phi][n_q][n_q], internal mode order
    int n_q, n_phi, NQP, batch, n_steps;
    int coeff_stride_q, coeff_stride_phi;
    const double *kv, *kq, *r, *astart;
    const float *s, *w;
    const double *q0, *v0;
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; const int *kperm; int *first_bad;
};

__host__ __device__ inline int small_h_stride(int n_q) { return n_q | 1; }      // odd row stride of H^n[k][.]
__host__ __device__ inline size_t small_smem_bytes(int n_q, int n_phi)
{
    return ((size_t)n_phi * n_q * small_h_stride(n_q) + (size_t)SM_WARPS * (32 + 32 + 32 * SM_TS)) * 4;
}

// HREG: N_q <= 16 and at most four (n, k) pairs per lane (N_phi N_q <= 128, e.g. 10 + 10 modes): the lane's rows of H live in registers
template <bool HREG>
__global__ void __launch_bounds__(SM_WARPS * 32) vk_small_kernel(const SmallArgs a)
{
    extern __shared__ __align__(16) float sm_smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nq = a.n_q, nphi = a.n_phi, hs = small_h_stride(nq);
    float *Hs = sm_smem;                                                   // [n_phi * n_q][hs]
    float *qs = Hs + (size_t)nphi * nq * hs + warp * (64 + 32 * SM_TS);    // [32] q^n as fp32
    float *es = qs + 32;                                                   // [32] eta_n
    float *ts = es + 32;                                                   // [n_phi][SM_TS]
    for (int i = tid; i < nphi * nq * nq; i += blockDim.x) { const int row = i / nq; Hs[(size_t)row * hs + (i - row * nq)] = __ldg(a.Hd + i); }
    __syncthreads();
    const int b = blockIdx.x * SM_WARPS + warp;
    if (b >= a.batch) return;
    const bool mine = lane < nq;
    const size_t co = (size_t)(a.coeff_stride_q ? b : 0) * a.NQP + lane;
    double q = 0.0, v = 0.0, kv = 0.0, kq = 0.0, r = 0.0, ast = 0.0, gn = 0.0; float wk = 0.f;
    if (mine) {
        q = a.q0[(size_t)b * a.NQP + lane]; v = a.v0[(size_t)b * a.NQP + lane];
        kv = a.kv[co]; kq = a.kq[co]; r = a.r[co]; ast = a.astart[co]; wk = a.w[co];
        if (a.fext) gn = a.gain[(size_t)b * a.NQP + lane];
    }
    const float sn = lane < nphi ? a.s[(size_t)(a.coeff_stride_phi ? b : 0) * nphi + lane] : 0.f;
    const int kp = mine ? a.kperm[lane] : 0;
    const int npairs = nphi * nq;
    float hreg[4][16]; int tpos[4];
    if (HREG) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int p = lane + 32 * j, nn = p / nq;
            tpos[j] = nn * SM_TS + (p - nn * nq);
#pragma unroll
            for (int rr = 0; rr < 16; ++rr) hreg[j][rr] = (p < npairs && rr < nq) ? Hs[(size_t)p * hs + rr] : 0.f;
        }
    }
    for (int i = lane; i < 64 + 32 * SM_TS; i += 32) qs[i] = 0.f;           // qs, es, ts of this warp: entries beyond the sizes stay zero
    __syncwarp();
    float oreg = 0.f;
    int bad = -1;
    float *out = a.out + (size_t)b * a.n_steps;
    for (int n = 0; n < a.n_steps; ++n) {
        const float x = (float)q;
        qs[lane] = x;
        __syncwarp();
        // a2: t[n][k] for the lane's pairs
        float qr[16];
        if (HREG) {
#pragma unroll
            for (int rr = 0; rr < 16; ++rr) qr[rr] = qs[rr];                   // 16 independent broadcast reads (zero beyond N_q)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
                for (int rr = 0; rr < 16; rr += 2) { acc0 = fmaf(hreg[j][rr], qr[rr], acc0); acc1 = fmaf(hreg[j][rr + 1], qr[rr + 1], acc1); }
                if (lane + 32 * j < npairs) ts[tpos[j]] = acc0 + acc1;
            }
        } else {
            for (int p = lane; p < npairs; p += 32) {
                const float *h = Hs + (size_t)p * hs;
                float acc0 = 0.f, acc1 = 0.f;
                int rr = 0;
#pragma unroll 4
                for (; rr + 1 < nq; rr += 2) { acc0 = fmaf(h[rr], qs[rr], acc0); acc1 = fmaf(h[rr + 1], qs[rr + 1], acc1); }
                if (rr < nq) acc0 = fmaf(h[rr], qs[rr], acc0);
                const int nn = p / nq;
                ts[nn * SM_TS + (p - nn * nq)] = acc0 + acc1;
            }
        }
        // a1 pickup + a6 write-out: placed here so that its shuffle chain runs while the t values settle in shared memory
        float o = wk * x, nr = x * x;
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) { o += __shfl_xor_sync(FLOW_FULL, o, m); nr += __shfl_xor_sync(FLOW_FULL, nr, m); }
        if (bad < 0 && !(isfinite(o) && isfinite(nr))) bad = n;
        if ((n & 31) == lane) oreg = o;
        if ((n & 31) == 31) out[n - 31 + lane] = oreg;
        if (a.traj && mine) a.traj[((size_t)b * a.n_steps + n) * nq + kp] = q;
        __syncwarp();
        // a3, a4: lane n
        if (lane < nphi) {
            const float *tr = ts + lane * SM_TS;
            float g0 = 0.f, g1 = 0.f;
            if (HREG) {                                                        // entries beyond N_q are zero on both sides
                float g2 = 0.f, g3 = 0.f;
#pragma unroll
                for (int k = 0; k < 16; k += 4) {
                    g0 = fmaf(qr[k], tr[k], g0); g1 = fmaf(qr[k + 1], tr[k + 1], g1); g2 = fmaf(qr[k + 2], tr[k + 2], g2); g3 = fmaf(qr[k + 3], tr[k + 3], g3);
                }
                g0 += g2; g1 += g3;
            } else {
                int k = 0;
#pragma unroll 4
                for (; k + 1 < nq; k += 2) { g0 = fmaf(qs[k], tr[k], g0); g1 = fmaf(qs[k + 1], tr[k + 1], g1); }
                if (k < nq) g0 = fmaf(qs[k], tr[k], g0);
            }
            es[lane] = sn * (g0 + g1);
        }
        __syncwarp();
        // force of mode `lane`, a5
        float f0 = 0.f, f1 = 0.f;
        if (mine) {
            int m = 0;
            float f2 = 0.f, f3 = 0.f;
            for (; m + 3 < nphi; m += 4) {                                     // four independent chains: the loads are all in flight
                f0 = fmaf(es[m], ts[m * SM_TS + lane], f0); f1 = fmaf(es[m + 1], ts[(m + 1) * SM_TS + lane], f1);
                f2 = fmaf(es[m + 2], ts[(m + 2) * SM_TS + lane], f2); f3 = fmaf(es[m + 3], ts[(m + 3) * SM_TS + lane], f3);
            }
            for (; m < nphi; ++m) f0 = fmaf(es[m], ts[m * SM_TS + lane], f0);
            f0 += f2; f1 += f3;
        }
        const double fd = (double)(f0 + f1);
        if (n == 0 && a.auto_start) v = (r != 0.0) ? ast * q + a.half_T2 * fd : 0.0;
        const double fe = a.fext ? (double)a.fext[(size_t)b * a.n_steps + n] * gn : 0.0;
        v = kv * v - kq * q + r * (fe - fd);
        q += v;
        __syncwarp();                                                      // qs, ts, es are rewritten in the next step
    }
    const int rem = a.n_steps & 31;
    if (rem && lane < rem) out[a.n_steps - rem + lane] = oreg;
    if (lane == 0) a.first_bad[b] = bad;
}

}  // namespace modal_dev
