// kernels.cuh -- hand-written sm_100a kernels of the modal hot path.
//
//   tension_kernel : MODAL_LINEAR / MODAL_TENSION, one warp per sample, state in registers
//                    (Eq. 8 + PAPER.md:153-167 Eq. 19-23).
//   vk_team_kernel : MODAL_VK, one persistent launch for the whole run.  A *team* of CTAs
//                    (one thread-block cluster, or every cluster of the grid) advances one
//                    sample; the packed coupling tensor is either resident in the team's
//                    shared memory or streamed from L2/HBM each step
//                    (Eq. 9-11, C eliminated by PAPER.md:283).
//
// Per step the vK kernel makes ONE pass over the symmetric-packed H:
//   t^n_k = sum_r H^n_kr q_r      (16x16 tiles of the lower triangle; each tile feeds the
//                                  row block AND, transposed, the column block)
//   G_n   = q . t^n ,  eta_n = s_n G_n ,  f_k = sum_n eta_n t^n_k
// q (x) q is never formed; reductions are warp shuffles; partial sums cross CTAs through
// distributed shared memory and, for grid-wide teams, one L2 exchange + grid barrier per step.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace modal_dev {
namespace cg = cooperative_groups;

constexpr int TILE = 16;            // tile edge of the packed H layout
constexpr int TILE_ELEMS = 256;
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

// ----------------------------------------------------------------------------------------
// von Karman team kernel
// ----------------------------------------------------------------------------------------

// One unit of work = tile-row I of in-plane mode n: tiles (I,0..I) of H^n.
struct __align__(16) VkUnit {
    int n;        // in-plane mode
    int I;        // tile row
    int nloc;     // n - first n of this cluster
    int tpoff;    // offset (floats) of this unit's partial-t vector in the CTA's tp buffer
    int gtile0;   // first tile in the global packed array: n * tiles_per_n + I(I+1)/2
    int ltile0;   // first tile in this CTA's resident shared-memory copy
    int pad0, pad1;
};

struct VkArgs {
    // coupling tensor + schedule
    const float *Ht;            // [n_phi][tiles_per_n][256] tile-packed lower triangle (see host_math.hpp)
    const VkUnit *units;        // all units, CTA-major then warp-major
    const int2 *warp_ptr;       // [sched_cta][NW] -> (first unit, count)
    const int2 *cta_ptr;        // [sched_cta]     -> (first unit, count)
    const int *nlo;             // [NCL+1] first in-plane mode of each cluster of a team
    int NQP, n_q, n_phi, tiles_per_n;
    int NLOC_MAX, CS, NCL, grid_team, resident;
    int max_cta_units, max_tp, max_cta_tiles;
    // per-sample coefficients
    int batch, n_steps;
    int coeff_stride_q, coeff_stride_phi;         // 0 = shared
    const double *kv, *kq, *r, *astart;           // [cb][NQP]
    const float *s, *w;                           // [cb][n_phi], [cb][NQP]
    const double *q0, *v0;                        // [batch][NQP]
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; int *first_bad;
    // grid-team exchange
    float *fbuf;                // [2][NCL][NQP]
    unsigned *counter;          // grid barrier arrivals (zeroed by the host before launch)
};

__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_gpu(unsigned *p, unsigned v)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Every CTA of the grid arrives once; returns when `target` arrivals are visible.
__device__ __forceinline__ void grid_barrier(unsigned *counter, unsigned target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        red_release_gpu(counter, 1u);
        while (ld_acquire_gpu(counter) < target) { }
        __threadfence();
    }
    __syncthreads();
}

// One tile-row: accumulates row and (transposed) column contributions of tiles (I, 0..I).
// tile: first tile of the row (shared or global), 64 float4 per tile.
// tp  : this unit's partial-t vector, (I+1)*16 floats, fully overwritten.
// returns the unit's contribution to G_n (all lanes).
template <bool GLOBAL>
__device__ __forceinline__ float tile_row_pass(const float4 *__restrict__ tile, const int I,
                                               const float *__restrict__ q32, float *__restrict__ tp,
                                               const int lane)
{
    const int r0 = lane >> 2, c0 = (lane & 3) * 4;
    const float qa = q32[I * TILE + r0], qb = q32[I * TILE + r0 + 8];
    const bool hi16 = lane & 16, hi8 = lane & 8;
    const int colsel = c0 + (hi16 ? 2 : 0) + (hi8 ? 1 : 0);
    float ra = 0.f, rb = 0.f;
#pragma unroll 4
    for (int J = 0; J <= I; ++J) {
        float4 ha, hb;
        if (GLOBAL) {
            ha = __ldg(tile + J * 64 + lane);
            hb = __ldg(tile + J * 64 + 32 + lane);
        } else {
            ha = tile[J * 64 + lane];
            hb = tile[J * 64 + 32 + lane];
        }
        const float4 qj = *reinterpret_cast<const float4 *>(q32 + J * TILE + c0);
        ra = fmaf(ha.x, qj.x, fmaf(ha.y, qj.y, fmaf(ha.z, qj.z, fmaf(ha.w, qj.w, ra))));
        rb = fmaf(hb.x, qj.x, fmaf(hb.y, qj.y, fmaf(hb.z, qj.z, fmaf(hb.w, qj.w, rb))));
        const float c_0 = fmaf(ha.x, qa, hb.x * qb), c_1 = fmaf(ha.y, qa, hb.y * qb);
        const float c_2 = fmaf(ha.z, qa, hb.z * qb), c_3 = fmaf(ha.w, qa, hb.w * qb);
        // transposing butterfly over the 8 row groups (lane bits 4,3,2)
        float k0 = hi16 ? c_2 : c_0, k1 = hi16 ? c_3 : c_1;
        const float s0 = hi16 ? c_0 : c_2, s1 = hi16 ? c_1 : c_3;
        k0 += __shfl_xor_sync(FULL, s0, 16);
        k1 += __shfl_xor_sync(FULL, s1, 16);
        float k = hi8 ? k1 : k0;
        const float s = hi8 ? k0 : k1;
        k += __shfl_xor_sync(FULL, s, 8);
        k += __shfl_xor_sync(FULL, k, 4);
        if (!(lane & 4)) tp[J * TILE + colsel] = k;
    }
    ra += __shfl_xor_sync(FULL, ra, 1); ra += __shfl_xor_sync(FULL, ra, 2);
    rb += __shfl_xor_sync(FULL, rb, 1); rb += __shfl_xor_sync(FULL, rb, 2);
    __syncwarp();
    float g = 0.f;
    if ((lane & 3) == 0) {
        tp[I * TILE + r0] += ra;
        tp[I * TILE + r0 + 8] += rb;
        g = fmaf(qa, ra, qb * rb);
    }
    g += __shfl_xor_sync(FULL, g, 4);
    g += __shfl_xor_sync(FULL, g, 8);
    g += __shfl_xor_sync(FULL, g, 16);
    g = __shfl_sync(FULL, g, 0);
    return 2.f * g;
}

// shared-memory carve-up (floats unless noted); must match vk_smem_bytes() on the host
struct VkSmem {
    float *q32, *eta, *gpart, *gu, *gx, *fpart, *fx, *tp;
    VkUnit *units;
    float4 *tiles;
};
__host__ __device__ inline size_t vk_align4(size_t x) { return (x + 3) & ~size_t(3); }
__host__ __device__ inline size_t vk_smem_floats(int NQP, int NLOC_MAX, int CS, int grid_team,
                                                 int max_cta_units, int max_tp)
{
    const size_t KS = (size_t)(NQP + CS - 1) / CS;
    size_t f = 0;
    f += vk_align4(NQP);                                   // q32
    f += vk_align4(NLOC_MAX) * 2;                          // eta, gpart
    f += vk_align4(max_cta_units);                         // gu
    f += vk_align4((size_t)CS * NLOC_MAX);                 // gx
    f += vk_align4(NQP);                                   // fpart
    f += vk_align4(grid_team ? (size_t)CS * KS : (size_t)CS * NQP);  // fx
    f += vk_align4(max_tp);                                // tp
    f += (size_t)max_cta_units * (sizeof(VkUnit) / 4);     // units
    return f;
}

template <bool RESIDENT>
__global__ void __launch_bounds__(512, 1) vk_team_kernel(const VkArgs a)
{
    extern __shared__ __align__(16) float smem[];
    cg::cluster_group cluster = cg::this_cluster();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NW = blockDim.x >> 5;
    const int CS = a.CS;
    const int rank = (int)cluster.block_rank();
    const int cl = blockIdx.x / CS;                         // cluster index in the grid
    const int tcl = a.grid_team ? cl : 0;                   // cluster index within the team
    const int scta = tcl * CS + rank;                       // CTA index in the schedule
    const int NQP = a.NQP, NLOC_MAX = a.NLOC_MAX;
    const int KS = (NQP + CS - 1) / CS;

    VkSmem S;
    {
        float *p = smem;
        S.q32 = p;   p += vk_align4(NQP);
        S.eta = p;   p += vk_align4(NLOC_MAX);
        S.gpart = p; p += vk_align4(NLOC_MAX);
        S.gu = p;    p += vk_align4(a.max_cta_units);
        S.gx = p;    p += vk_align4((size_t)CS * NLOC_MAX);
        S.fpart = p; p += vk_align4(NQP);
        S.fx = p;    p += vk_align4(a.grid_team ? (size_t)CS * KS : (size_t)CS * NQP);
        S.tp = p;    p += vk_align4(a.max_tp);
        S.units = reinterpret_cast<VkUnit *>(p); p += (size_t)a.max_cta_units * (sizeof(VkUnit) / 4);
        S.tiles = reinterpret_cast<float4 *>(p);
    }
    const int2 cu = a.cta_ptr[scta];                        // this CTA's units
    const int2 wu = a.warp_ptr[scta * NW + warp];           // this warp's units
    const int nlo = a.nlo[tcl], nloc_cnt = a.nlo[tcl + 1] - nlo;
    for (int u = tid; u < cu.y; u += blockDim.x) S.units[u] = a.units[cu.x + u];
    __syncthreads();
    if (RESIDENT) {  // copy this CTA's tiles into shared memory once
        for (int u = 0; u < cu.y; ++u) {
            const VkUnit un = S.units[u];
            const float4 *src = reinterpret_cast<const float4 *>(a.Ht) + (size_t)un.gtile0 * 64;
            float4 *dst = S.tiles + (size_t)un.ltile0 * 64;
            for (int i = tid; i < (un.I + 1) * 64; i += blockDim.x) dst[i] = __ldg(src + i);
        }
    }
    const float4 *Hg = reinterpret_cast<const float4 *>(a.Ht);
    unsigned epoch = 0;
    const bool out_cta = (rank == 0) && (a.grid_team ? cl == 0 : true);
    const int b_begin = a.grid_team ? 0 : cl;
    const int b_step = a.grid_team ? 1 : (int)(gridDim.x / CS);

    for (int b = b_begin; b < a.batch; b += b_step) {
        // ---- per-sample state (thread k owns mode k) ----
        double q = 0, v = 0, kv = 0, kq = 0, r = 0, ast = 0, gain = 0;
        float wk = 0;
        const size_t coq = (size_t)(a.coeff_stride_q ? b : 0) * NQP;
        const float *sb = a.s + (size_t)(a.coeff_stride_phi ? b : 0) * a.n_phi;
        if (tid < NQP) {
            q = a.q0[(size_t)b * NQP + tid]; v = a.v0[(size_t)b * NQP + tid];
            kv = a.kv[coq + tid]; kq = a.kq[coq + tid]; r = a.r[coq + tid]; ast = a.astart[coq + tid];
            wk = a.w[coq + tid];
            gain = a.fext ? a.gain[(size_t)b * NQP + tid] : 0.0;
            S.q32[tid] = (float)q;
        }
        float oreg = 0.f;
        int bad = -1;
        float *out = a.out + (size_t)b * a.n_steps;
        __syncthreads();

        for (int n = 0; n < a.n_steps; ++n) {
            // ---- a1 pickup + a6 write-out (last warp of the output CTA) ----
            if (out_cta && warp == NW - 1) {
                float o = 0.f, nrm = 0.f;
                for (int k = lane; k < NQP; k += 32) {
                    const float qk = S.q32[k];
                    o = fmaf(a.w[coq + k], qk, o);
                    nrm = fmaf(qk, qk, nrm);
                }
#pragma unroll
                for (int m = 16; m >= 1; m >>= 1) {
                    o += __shfl_xor_sync(FULL, o, m);
                    nrm += __shfl_xor_sync(FULL, nrm, m);
                }
                if (bad < 0 && !(isfinite(o) && isfinite(nrm))) bad = n;
                if ((n & 31) == lane) oreg = o;
                if ((n & 31) == 31) out[n - 31 + lane] = oreg;
            }
            if (out_cta && a.traj && tid < a.n_q)
                a.traj[((size_t)b * a.n_steps + n) * a.n_q + tid] = q;

            // ---- a2+a3 phase A: one pass over this warp's tile rows ----
            for (int u = wu.x - cu.x; u < wu.x - cu.x + wu.y; ++u) {
                const VkUnit un = S.units[u];
                const float4 *tile = RESIDENT ? S.tiles + (size_t)un.ltile0 * 64
                                              : Hg + (size_t)un.gtile0 * 64;
                const float g = tile_row_pass<!RESIDENT>(tile, un.I, S.q32, S.tp + un.tpoff, lane);
                if (lane == 0) S.gu[u] = g;
            }
            __syncthreads();
            // per-CTA partial G for each in-plane mode of the cluster, pushed to every CTA
            if (tid < nloc_cnt) {
                float g = 0.f;
                for (int u = 0; u < cu.y; ++u)
                    if (S.units[u].nloc == tid) g += S.gu[u];
                for (int d = 0; d < CS; ++d)
                    cluster.map_shared_rank(S.gx, d)[rank * NLOC_MAX + tid] = g;
            }
            cluster.sync();
            if (tid < nloc_cnt) {
                float G = 0.f;
                for (int d = 0; d < CS; ++d) G += S.gx[d * NLOC_MAX + tid];
                S.eta[tid] = sb[nlo + tid] * G;                     // eta_n = s_n G_n
            }
            __syncthreads();
            // ---- phase B: f_k partial of this CTA ----
            float f = 0.f;
            if (tid < NQP) {
                for (int u = 0; u < cu.y; ++u) {
                    const VkUnit un = S.units[u];
                    if (tid < (un.I + 1) * TILE) f = fmaf(S.eta[un.nloc], S.tp[un.tpoff + tid], f);
                }
            }
            if (!a.grid_team) {
                // all-to-all inside the cluster
                if (tid < NQP)
                    for (int d = 0; d < CS; ++d)
                        cluster.map_shared_rank(S.fx, d)[rank * NQP + tid] = f;
                cluster.sync();
                f = 0.f;
                if (tid < NQP)
                    for (int d = 0; d < CS; ++d) f += S.fx[d * NQP + tid];
            } else {
                // reduce-scatter inside the cluster, then one L2 exchange across clusters
                if (tid < NQP) {
                    const int d = tid / KS;
                    cluster.map_shared_rank(S.fx, d)[rank * KS + (tid - d * KS)] = f;
                }
                cluster.sync();
                float *fb = a.fbuf + ((size_t)(epoch & 1) * a.NCL + cl) * NQP;
                if (tid < KS && rank * KS + tid < NQP) {
                    float fs = 0.f;
                    for (int d = 0; d < CS; ++d) fs += S.fx[d * KS + tid];
                    __stcg(fb + rank * KS + tid, fs);
                }
                ++epoch;
                grid_barrier(a.counter, epoch * gridDim.x);
                f = 0.f;
                if (tid < NQP) {
                    const float *fr = a.fbuf + (size_t)((epoch - 1) & 1) * a.NCL * NQP + tid;
                    for (int c = 0; c < a.NCL; ++c) f += __ldcg(fr + (size_t)c * NQP);
                }
            }
            // ---- a5 linear update (fp64, delta form) ----
            if (tid < NQP) {
                const double fd = (double)f;
                if (n == 0 && a.auto_start) v = (r != 0.0) ? ast * q + a.half_T2 * fd : 0.0;
                const double fe = a.fext ? (double)a.fext[(size_t)b * a.n_steps + n] * gain : 0.0;
                v = kv * v - kq * q + r * (fe - fd);
                q += v;
                S.q32[tid] = (float)q;
            }
            __syncthreads();
        }
        if (out_cta && warp == NW - 1) {
            const int rem = a.n_steps & 31;
            if (rem && lane < rem) out[a.n_steps - rem + lane] = oreg;
            if (lane == 0) a.first_bad[b] = bad;
        }
        __syncthreads();
    }
    cluster.sync();   // no CTA may exit while a peer can still write its shared memory
}

}  // namespace modal_dev
