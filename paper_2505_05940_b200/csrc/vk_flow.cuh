// vk_flow.cuh -- MODAL_VK time loop as ONE persistent sm_100a kernel.
//
// A *team* of G CTAs (one per SM) advances one sample at a time; NT teams run side by side on
// different samples.  Each CTA owns a contiguous range of the symmetric-packed coupling tensor
// (flow_schedule.hpp): the leading part of the range stays resident in shared memory for the
// whole run, the rest is streamed every time step from L2/HBM by a producer warp with TMA bulk
// copies (cp.async.bulk + mbarrier) into a ring of slots; the ring keeps filling while the team
// exchanges data, so the stream never stops at a step boundary.
//
// Per time step (Eq. 9 with C eliminated by PAPER.md:283; Eq. 20-23 / 16-19):
//   A   every consumer warp makes ONE pass over its units:  t^n_k += H^n_kr q_r  for the row block
//       and, transposed, the column blocks of each stored tile; q (x) q is never formed.
//   B1  G_n = q . t^n  per in-plane mode; modes split over several CTAs all-gather their partial
//       G_n through L2;  eta_n = s_n G_n.
//   B2  partial force  f_k = sum_n eta_n t^n_k  of this CTA, published to L2.
//   C   the CTA that owns mode k sums the G partials in rank order (deterministic), applies the
//       fp64 delta-form update and publishes q_k^{n+1}.
//   D   every CTA gathers q^{n+1}.
// Cross-CTA data travels as 64-bit words {fp32 value, 32-bit epoch}: a reader polls the word until
// the epoch matches, so there is no grid barrier, no atomic and no fence on the step path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace modal_dev {

constexpr unsigned FLOW_FULL = 0xffffffffu;

struct FlowArgs {
    const float *Hf;            // flow-tile-packed coupling tensor
    const int *sched;           // [G][sched_stride]
    int sched_stride;
    int off_units, off_ltile, off_pieces, off_pu, off_kbptr, off_kblist;
    int G, NT, NW, NS, slot_tiles;
    int direct;                 // 1: units that are not resident are read straight from L2/HBM by the consumers (no ring)
    int NQP, n_q, n_phi, nb;
    int U_max, tp_max, NLOC_MAX, res_tiles, slice_max, MS;
    int batch, n_steps;
    int coeff_stride_q, coeff_stride_phi;         // 0 = shared coefficients
    const double *kv, *kq, *r, *astart;           // [cb][NQP]
    const float *s, *w;                           // [cb][n_phi], [cb][NQP]
    const double *q0, *v0;                        // [batch][NQP]
    int auto_start; double half_T2;
    const float *fext; const double *gain;
    float *out; double *traj; const int *kperm; int *first_bad;   // kperm[k]: user index of internal mode k (trajectory rows)
    unsigned long long *fx;     // [NT][G][NQP]   partial forces
    unsigned long long *gx;     // [NT][n_phi][MS] partial G_n of shared modes
    unsigned long long *qx;     // [NT][FLOW_QREP][NQP]  new state
    int *timeout_flag;          // per plan: set when a bounded wait gave up
    long long *timing;          // optional [G*NT][8]: cycles in phases A, B1, B2+C+D, total (MODAL_FLOW_TIMING)
};

// ---- tagged 64-bit words through L2 ----------------------------------------------------------
__device__ __forceinline__ void st_tag(unsigned long long *p, float v, unsigned epoch)
{
    const unsigned long long w = ((unsigned long long)epoch << 32) | (unsigned long long)__float_as_uint(v);
    asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
// Every wait is bounded (~1-2 s): a waiter that gives up raises the CTA's abort word, after which all waits
// of the CTA fall through and the step loop ends; the CTA then raises the plan's timeout flag, so a broken
// exchange (e.g. a team that is not co-resident) ends in an error code instead of a hung device.
__device__ __forceinline__ float ld_tag(const unsigned long long *p, unsigned epoch, volatile int *abortp)
{
    unsigned long long w;
    unsigned spins = 0;
    do {
        asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(w) : "l"(p) : "memory");
        if ((unsigned)(w >> 32) == epoch) break;
        if ((++spins & 1023u) == 0 && (*abortp || spins > (1u << 21))) { *abortp = 1; break; }
    } while (true);
    return __uint_as_float((unsigned)w);
}

// two adjacent tagged words with one 16-byte load (each 8-byte half is single-copy atomic)
__device__ __forceinline__ float2 ld_tag2(const unsigned long long *p, unsigned epoch, volatile int *abortp)
{
    unsigned long long w0, w1;
    unsigned spins = 0;
    do {
        asm volatile("ld.relaxed.gpu.global.v2.b64 {%0, %1}, [%2];" : "=l"(w0), "=l"(w1) : "l"(p) : "memory");
        if ((unsigned)(w0 >> 32) == epoch && (unsigned)(w1 >> 32) == epoch) break;
        if ((++spins & 1023u) == 0 && (*abortp || spins > (1u << 21))) { *abortp = 1; break; }
    } while (true);
    return make_float2(__uint_as_float((unsigned)w0), __uint_as_float((unsigned)w1));
}
// sum of the tagged words p[i * stride], i = 0 .. cnt-1 (cnt <= 8), all loads in flight together;
// words that are not there yet are polled again.  Fixed summation order.
__device__ __forceinline__ float ld_tag_sum8(const unsigned long long *p, size_t stride, int cnt, unsigned epoch,
                                            volatile int *abortp)
{
    float v[8];
    unsigned pend = cnt >= 8 ? 0xffu : ((1u << cnt) - 1u), spins = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = 0.f;
    while (pend) {
        unsigned long long w[8];
#pragma unroll
        for (int i = 0; i < 8; ++i)
            if (pend >> i & 1) asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(w[i]) : "l"(p + i * stride) : "memory");
#pragma unroll
        for (int i = 0; i < 8; ++i)
            if ((pend >> i & 1) && (unsigned)(w[i] >> 32) == epoch) { v[i] = __uint_as_float((unsigned)w[i]); pend &= ~(1u << i); }
        if (pend && (++spins & 1023u) == 0 && (*abortp || spins > (1u << 21))) { *abortp = 1; break; }
    }
    return ((v[0] + v[1]) + (v[2] + v[3])) + ((v[4] + v[5]) + (v[6] + v[7]));
}
constexpr int FLOW_QREP = 4;     // replicas of the published state: spreads the pollers over L2 slices

// ---- mbarrier / TMA bulk copy ----------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, volatile int *abortp)
{
    uint32_t ok;
    unsigned spins = 0;
    const long long t0 = clock64();
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (!ok && (++spins & 63u) == 0 && (*abortp || clock64() - t0 > 3000000000LL)) { *abortp = 1; break; }
    } while (!ok);
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ int bar_consumers_or(int nthreads, int pred)
{
    int r;
    asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.s32 p, %2, 0;\n\tbar.red.or.pred q, 1, %1, p;\n\tselp.s32 %0, 1, 0, q;\n\t}"
                 : "=r"(r) : "r"(nthreads), "r"(pred) : "memory");
    return r;
}
__device__ __forceinline__ void bar_consumers(int nthreads)
{
    asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

// row sums of a unit: transposing butterfly over the 16 column lanes (bits 3,2,1 of j), then bit 0;
// writes the 16 row sums after the column groups and returns the unit's share of G_n
__device__ __forceinline__ float flow_unit_rows(float a0, float a1, float a2, float a3, float a4, float a5, float a6, float a7,
                                                const int I, const int nt, const float *__restrict__ q32,
                                                float *__restrict__ tp, const int lane)
{
    const int j = lane & 15, half = lane >> 4;
    const bool b8 = j & 8, b4 = j & 4, b2 = j & 2;
    float v0 = (b8 ? a4 : a0) + __shfl_xor_sync(FLOW_FULL, b8 ? a0 : a4, 8);
    float v1 = (b8 ? a5 : a1) + __shfl_xor_sync(FLOW_FULL, b8 ? a1 : a5, 8);
    float v2 = (b8 ? a6 : a2) + __shfl_xor_sync(FLOW_FULL, b8 ? a2 : a6, 8);
    float v3 = (b8 ? a7 : a3) + __shfl_xor_sync(FLOW_FULL, b8 ? a3 : a7, 8);
    float w0 = (b4 ? v2 : v0) + __shfl_xor_sync(FLOW_FULL, b4 ? v0 : v2, 4);
    float w1 = (b4 ? v3 : v1) + __shfl_xor_sync(FLOW_FULL, b4 ? v1 : v3, 4);
    float x = (b2 ? w1 : w0) + __shfl_xor_sync(FLOW_FULL, b2 ? w0 : w1, 2);
    x += __shfl_xor_sync(FLOW_FULL, x, 1);
    const int row = half * 8 + (b2 ? 1 : 0) + (b4 ? 2 : 0) + (b8 ? 4 : 0);
    float g = 0.f;
    if (!(j & 1)) {
        tp[nt * 16 + row] = x;
        g = q32[I * 16 + row] * x;
    }
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) g += __shfl_xor_sync(FLOW_FULL, g, m);
    return 2.f * g;
}

// ---- one unit: tiles (I, J0 .. J0+nt-1) of one H^n -------------------------------------------
// tile : first tile of the unit in shared memory, 64 float4 per tile (flow layout)
// tp   : the unit's output: nt*16 column sums (block J0+t at tp[t*16..]) then 16 row sums
// returns the unit's contribution to G_n = q^T H^n q (all lanes)
__device__ __forceinline__ float flow_unit(const float4 *__restrict__ tile, const int I, const int J0, const int nt,
                                           const float *__restrict__ q32, float *__restrict__ tp, const int lane)
{
    const int j = lane & 15, half = lane >> 4;
    const float4 qa = *reinterpret_cast<const float4 *>(q32 + I * 16 + half * 8);
    const float4 qb = *reinterpret_cast<const float4 *>(q32 + I * 16 + half * 8 + 4);
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f, a5 = 0.f, a6 = 0.f, a7 = 0.f;
    const float *qj = q32 + J0 * 16 + j;
#pragma unroll 2
    for (int t = 0; t < nt; ++t) {
        const float4 h0 = tile[t * 64 + lane];
        const float4 h1 = tile[t * 64 + 32 + lane];
        const float x = qj[t * 16];
        float c = h0.x * qa.x;
        c = fmaf(h0.y, qa.y, c); c = fmaf(h0.z, qa.z, c); c = fmaf(h0.w, qa.w, c);
        c = fmaf(h1.x, qb.x, c); c = fmaf(h1.y, qb.y, c); c = fmaf(h1.z, qb.z, c); c = fmaf(h1.w, qb.w, c);
        a0 = fmaf(h0.x, x, a0); a1 = fmaf(h0.y, x, a1); a2 = fmaf(h0.z, x, a2); a3 = fmaf(h0.w, x, a3);
        a4 = fmaf(h1.x, x, a4); a5 = fmaf(h1.y, x, a5); a6 = fmaf(h1.z, x, a6); a7 = fmaf(h1.w, x, a7);
        c += __shfl_xor_sync(FLOW_FULL, c, 16);
        if (half == 0) tp[t * 16 + j] = c;
    }
    return flow_unit_rows(a0, a1, a2, a3, a4, a5, a6, a7, I, nt, q32, tp, lane);
}

// Same unit with the tiles read straight from global memory (L2): all tiles of the unit (<= 16 LDG.128 per lane) are
// issued before they are consumed; with 16 warps that keeps up to ~128 KB per SM in flight, which measures
// ~20 TB/s from L2 on B200, against ~4 TB/s for the cp.async.bulk ring (profiles/r1_c4_b1.md).
__device__ __forceinline__ float flow_unit_direct(const float4 *__restrict__ tile, const int I, const int J0, const int nt,
                                                  const float *__restrict__ q32, float *__restrict__ tp, const int lane)
{
    const int j = lane & 15, half = lane >> 4;
    const float4 qa = *reinterpret_cast<const float4 *>(q32 + I * 16 + half * 8);
    const float4 qb = *reinterpret_cast<const float4 *>(q32 + I * 16 + half * 8 + 4);
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f, a5 = 0.f, a6 = 0.f, a7 = 0.f;
    const float *qj = q32 + J0 * 16 + j;
    float4 h[16];                                            // the whole unit (<= 8 tiles) in flight
#pragma unroll
    for (int u = 0; u < 8; ++u)
        if (u < nt) { h[2 * u] = __ldcg(tile + u * 64 + lane); h[2 * u + 1] = __ldcg(tile + u * 64 + 32 + lane); }
#pragma unroll
    for (int u = 0; u < 8; ++u)
        if (u < nt) {
            const float4 h0 = h[2 * u], h1 = h[2 * u + 1];
            const float x = qj[u * 16];
            float c = h0.x * qa.x;
            c = fmaf(h0.y, qa.y, c); c = fmaf(h0.z, qa.z, c); c = fmaf(h0.w, qa.w, c);
            c = fmaf(h1.x, qb.x, c); c = fmaf(h1.y, qb.y, c); c = fmaf(h1.z, qb.z, c); c = fmaf(h1.w, qb.w, c);
            a0 = fmaf(h0.x, x, a0); a1 = fmaf(h0.y, x, a1); a2 = fmaf(h0.z, x, a2); a3 = fmaf(h0.w, x, a3);
            a4 = fmaf(h1.x, x, a4); a5 = fmaf(h1.y, x, a5); a6 = fmaf(h1.z, x, a6); a7 = fmaf(h1.w, x, a7);
            c += __shfl_xor_sync(FLOW_FULL, c, 16);
            if (half == 0) tp[u * 16 + j] = c;
        }
    return flow_unit_rows(a0, a1, a2, a3, a4, a5, a6, a7, I, nt, q32, tp, lane);
}

__host__ __device__ inline size_t flow_align(size_t x, size_t a) { return (x + a - 1) / a * a; }

// shared-memory carve-up in bytes; the host uses the same function to size the launch
struct FlowSmem {
    size_t bars, q32, eta, gu, fpart, sq, sv, tp, sched, ring, res, total;
};
__host__ __device__ inline FlowSmem flow_smem_layout(int NS, int slot_tiles, int NQP, int NLOC_MAX, int U_max,
                                                     int slice_max, int tp_max, int sched_stride, int res_tiles, bool single_cta = true)
{
    FlowSmem L;
    size_t o = 0;
    L.bars = o;  o += flow_align((size_t)3 * (NS > 0 ? NS : 1) * 8 + 16, 16);   // full, empty, done[], abort
    L.q32 = o;   o += flow_align((size_t)NQP * 4, 16);
    L.eta = o;   o += flow_align((size_t)NLOC_MAX * 4, 16);
    L.gu = o;    o += flow_align((size_t)U_max * 4, 16);
    L.fpart = o; o += single_cta ? flow_align((size_t)NQP * 4, 16) : 0;      // the force of a one-CTA team; teams exchange it through L2 (1.6 KB that make C4's 207 tiles per CTA resident)
    L.sq = o;    o += flow_align((size_t)slice_max * 8, 16);
    L.sv = o;    o += flow_align((size_t)slice_max * 8, 16);
    L.tp = o;    o += flow_align((size_t)tp_max * 4, 16);
    L.sched = o; o += flow_align((size_t)sched_stride * 4, 16);
    o = flow_align(o, 128);
    L.ring = o;  o += (size_t)NS * slot_tiles * 1024;
    L.res = o;   o += (size_t)res_tiles * 1024;
    L.total = o;
    return L;
}

// RING = true: 16 consumer warps + the TMA producer warp; false: consumers only (resident and direct units)
template <bool RING>
__global__ void __launch_bounds__(RING ? 544 : 512, 1) vk_flow_kernel(const FlowArgs a)
{
    extern __shared__ __align__(128) unsigned char flow_smem[];
    unsigned char *smem = flow_smem;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NW = a.NW, NC = NW * 32, G = a.G, NQP = a.NQP;
    const int team = blockIdx.x / G, rank = blockIdx.x - team * G;
    const FlowSmem L = flow_smem_layout(a.NS, a.slot_tiles, NQP, a.NLOC_MAX, a.U_max, a.slice_max, a.tp_max,
                                        a.sched_stride, a.res_tiles, a.G == 1);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + L.bars);
    volatile unsigned *done = reinterpret_cast<volatile unsigned *>(bars + 2 * (a.NS > 0 ? a.NS : 1));   // uses consumed per slot
    volatile int *s_abort = reinterpret_cast<volatile int *>(done + 2 * (a.NS > 0 ? a.NS : 1));
    float *q32 = reinterpret_cast<float *>(smem + L.q32);
    float *eta = reinterpret_cast<float *>(smem + L.eta);
    float *gu = reinterpret_cast<float *>(smem + L.gu);
    float *fpart = reinterpret_cast<float *>(smem + L.fpart);
    double *sq = reinterpret_cast<double *>(smem + L.sq);
    double *sv = reinterpret_cast<double *>(smem + L.sv);
    float *tp = reinterpret_cast<float *>(smem + L.tp);
    int *sch = reinterpret_cast<int *>(smem + L.sched);
    float4 *ring = reinterpret_cast<float4 *>(smem + L.ring);
    float4 *res = reinterpret_cast<float4 *>(smem + L.res);

    for (int i = tid; i < a.sched_stride; i += blockDim.x) sch[i] = a.sched[(size_t)rank * a.sched_stride + i];
    if (tid == 0) {
        for (int s = 0; s < a.NS; ++s) { mbar_init(smem_u32(bars + s), 1); mbar_init(smem_u32(bars + a.NS + s), 1); done[s] = 0; }
        *s_abort = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int U = sch[0], R = sch[1], NLOC = sch[2], slice0 = sch[4], slice_len = sch[5];
    const int S = a.direct ? 0 : U - R;                        // units per time step that go through the TMA ring
    const int4 *units = reinterpret_cast<const int4 *>(sch + a.off_units);
    const int *ltile = sch + a.off_ltile;
    const int4 *pieces = reinterpret_cast<const int4 *>(sch + a.off_pieces);
    const int *pu = sch + a.off_pu, *kbptr = sch + a.off_kbptr, *kblist = sch + a.off_kblist;
    const float4 *Hg = reinterpret_cast<const float4 *>(a.Hf);
    // resident part of this CTA's range: loaded once
    for (int u = 0; u < R; ++u) {
        const int4 un = units[u];
        const int ntl = (un.x >> 16) & 0xff;
        const float4 *src = Hg + (size_t)un.w * 64;
        float4 *dst = res + (size_t)ltile[u] * 64;
        for (int i = tid; i < ntl * 64; i += blockDim.x) dst[i] = __ldg(src + i);
    }
    __syncthreads();
    const int my_samples = team < a.batch ? (a.batch - team + a.NT - 1) / a.NT : 0;
    const long long total_steps = (long long)my_samples * a.n_steps;

    if (RING && warp == NW) {
        // ---------------- producer: TMA bulk copies of the streamed units, step after step --------
        // Lane l owns ring slot l (NS <= 32): the items of a slot are it = l, l+NS, l+2NS, ...  Every lane
        // runs a non-blocking state machine (test_wait, then issue), so 32 copies are prepared side by
        // side and no lane ever waits on another.
        if (S > 0 && lane < a.NS) {
            const long long total_items = total_steps * S;
            const int step_u = a.NS % S;
            long long it = lane;
            int ui = lane % S;                                  // it % S
            unsigned use = 0, idle = 0;
            const uint32_t full = smem_u32(bars + lane), empty = smem_u32(bars + a.NS + lane);
            const uint32_t dst = smem_u32(ring + (size_t)lane * a.slot_tiles * 64);
            long long t0 = clock64();
            while (it < total_items) {
                uint32_t ok;
                asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                             "selp.u32 %0, 1, 0, p;\n\t}"
                             : "=r"(ok) : "r"(empty), "r"((use & 1) ^ 1) : "memory");
                if (ok) {
                    const int4 un = units[R + ui];
                    const uint32_t bytes = (uint32_t)((un.x >> 16) & 0xff) * 1024u;
                    mbar_expect_tx(full, bytes);
                    tma_bulk_g2s(dst, Hg + (size_t)un.w * 64, bytes, full);
                    it += a.NS; ++use; idle = 0;
                    ui += step_u; if (ui >= S) ui -= S;
                } else if ((++idle & 255u) == 0) {
                    if (idle == 256) t0 = clock64();
                    if (*s_abort || clock64() - t0 > 3000000000LL) { *s_abort = 1; break; }
                }
            }
        }
        return;
    }

    // ---------------- consumers ---------------------------------------------------------------
    unsigned epoch = 0;
    unsigned ring_pos = 0, ring_use = 0;                       // ring slot / use count at the start of the step
    unsigned long long *fx = a.fx + (size_t)team * G * NQP;
    unsigned long long *gx = a.gx + (size_t)team * a.n_phi * a.MS;
    unsigned long long *qx = a.qx + (size_t)team * FLOW_QREP * NQP;
    const unsigned long long *qx_mine = qx + (size_t)(rank % FLOW_QREP) * NQP;
    const bool out_cta = rank == 0;

    for (int b = team; b < a.batch; b += a.NT) {
        const size_t coq = (size_t)(a.coeff_stride_q ? b : 0) * NQP;
        const float *sb = a.s + (size_t)(a.coeff_stride_phi ? b : 0) * a.n_phi;
        for (int k = tid; k < NQP; k += NC) q32[k] = (float)a.q0[(size_t)b * NQP + k];
        for (int j = tid; j < slice_len; j += NC) {
            sq[j] = a.q0[(size_t)b * NQP + slice0 + j];
            sv[j] = a.v0[(size_t)b * NQP + slice0 + j];
        }
        float oreg = 0.f;
        int bad = -1;
        float *out = a.out + (size_t)b * a.n_steps;
        bar_consumers(NC);

        for (int n = 0; n < a.n_steps; ++n) {
            ++epoch;
            long long tk0 = 0, tk1 = 0, tk2 = 0, tkb = 0, tkc = 0;
            if (a.timing && tid == 0) tk0 = clock64();
            // ---- a1 pickup + a6 write-out (last consumer warp of rank 0) ----
            if (out_cta && warp == NW - 1) {
                float o = 0.f, nrm = 0.f;
                for (int k = lane; k < NQP; k += 32) {
                    const float qk = q32[k];
                    o = fmaf(a.w[coq + k], qk, o);
                    nrm = fmaf(qk, qk, nrm);
                }
#pragma unroll
                for (int m = 16; m >= 1; m >>= 1) {
                    o += __shfl_xor_sync(FLOW_FULL, o, m);
                    nrm += __shfl_xor_sync(FLOW_FULL, nrm, m);
                }
                if (bad < 0 && !(isfinite(o) && isfinite(nrm))) bad = n;
                if ((n & 31) == lane) oreg = o;
                if ((n & 31) == 31) out[n - 31 + lane] = oreg;
            }
            if (a.traj)
                for (int j = tid; j < slice_len; j += NC)
                    if (slice0 + j < a.n_q) a.traj[((size_t)b * a.n_steps + n) * a.n_q + a.kperm[slice0 + j]] = sq[j];

            // ---- A: one pass over this warp's units ----
            for (int u = warp; u < U; u += NW) {
                const int4 un = units[u];
                const int I = (un.x >> 8) & 0xff, ntl = (un.x >> 16) & 0xff;
                const float4 *tile;
                int slot = 0;
                unsigned use = 0;
                if (u < R) tile = res + (size_t)ltile[u] * 64;
                else if (a.direct) {
                    const float g = flow_unit_direct(Hg + (size_t)un.w * 64, I, un.y, ntl, q32, tp + un.z, lane);
                    if (lane == 0) gu[u] = g;
                    continue;
                } else {
                    const unsigned x = ring_pos + (unsigned)(u - R);
                    slot = (int)(x % (unsigned)a.NS);
                    use = ring_use + x / (unsigned)a.NS;
                    // a parity wait is only valid one phase ahead: first wait until the slot's previous
                    // use has been consumed (another warp may still be working on it)
                    if (lane == 0) {
                        unsigned spins = 0;
                        while (done[slot] != use) if ((++spins & 1023u) == 0 && (*s_abort || spins > (1u << 24))) { *s_abort = 1; break; }
                    }
                    __syncwarp();
                    mbar_wait(smem_u32(bars + slot), use & 1, s_abort);
                    tile = ring + (size_t)slot * a.slot_tiles * 64;
                }
                const float g = flow_unit(tile, I, un.y, ntl, q32, tp + un.z, lane);
                if (lane == 0) gu[u] = g;
                if (u >= R) {
                    __syncwarp();
                    if (lane == 0) { done[slot] = use + 1; mbar_arrive(smem_u32(bars + a.NS + slot)); }
                }
            }
            if (S > 0) {
                const unsigned x = ring_pos + (unsigned)S;
                ring_pos = x % (unsigned)a.NS; ring_use += x / (unsigned)a.NS;
            }
            if (bar_consumers_or(NC, *s_abort)) break;      // uniform: nobody is left behind at a barrier
            if (a.timing && tid == 0) tk1 = clock64();

            // ---- B1: G_n per piece (fixed summation order), all-gather over the sharers ----
            for (int p = warp; p < NLOC; p += NW) {
                const int4 pc = pieces[p];                        // {n, first sharer, sharers, my slot}
                float g = 0.f;
                for (int u = pu[p] + lane; u < pu[p + 1]; u += 32) g += gu[u];
#pragma unroll
                for (int m = 16; m >= 1; m >>= 1) g += __shfl_xor_sync(FLOW_FULL, g, m);
                float Gn = g;
                if (pc.z > 1) {
                    unsigned long long *slot0 = gx + (size_t)pc.x * a.MS;
                    if (lane == 0) st_tag(slot0 + pc.w, g, epoch);
                    Gn = 0.f;
                    for (int base = 0; base < pc.z; base += 32) {          // slot order: same sum on every sharer
                        float part = 0.f;
                        if (base + lane < pc.z) part = base + lane == pc.w ? g : ld_tag(slot0 + base + lane, epoch, s_abort);
                        const int cnt = min(32, pc.z - base);
                        for (int s = 0; s < cnt; ++s) Gn += __shfl_sync(FLOW_FULL, part, s);
                    }
                }
                if (lane == 0) eta[p] = sb[pc.x] * Gn;           // eta_n = s_n G_n
            }
            bar_consumers(NC);
            if (a.timing && tid == 0) tk2 = clock64();

            // ---- B2: partial force of this CTA ----
            for (int k = tid; k < NQP; k += NC) {
                const int K = k >> 4, kk = k & 15;
                float f0 = 0.f, f1 = 0.f;
                int e = kbptr[K];
                const int e1 = kbptr[K + 1];
                for (; e + 1 < e1; e += 2) {
                    const int x0 = kblist[e], x1 = kblist[e + 1];
                    f0 = fmaf(eta[(unsigned)x0 >> 24], tp[(x0 & 0xffffff) + kk], f0);
                    f1 = fmaf(eta[(unsigned)x1 >> 24], tp[(x1 & 0xffffff) + kk], f1);
                }
                if (e < e1) { const int x0 = kblist[e]; f0 = fmaf(eta[(unsigned)x0 >> 24], tp[(x0 & 0xffffff) + kk], f0); }
                const float f = f0 + f1;
                if (G > 1) st_tag(fx + (size_t)rank * NQP + k, f, epoch);
                else fpart[k] = f;
            }
            if (a.timing && tid == 0) tkb = clock64();
            // ---- C: owner of mode k: rank-ordered sum, a5 linear update (fp64, delta form) ----
            if (G > 1) {
                for (int j = warp; j < slice_len; j += NW) {
                    const int k = slice0 + j;
                    float f = 0.f;
                    for (int c0 = lane; c0 < G; c0 += 256)          // 8 partials per lane in flight
                        f += ld_tag_sum8(fx + (size_t)c0 * NQP + k, (size_t)32 * NQP, min(8, (G - c0 + 31) / 32), epoch, s_abort);
#pragma unroll
                    for (int m = 16; m >= 1; m >>= 1) f += __shfl_xor_sync(FLOW_FULL, f, m);
                    if (lane == 0) {
                        const double fd = (double)f, r = a.r[coq + k];
                        double q = sq[j], v = sv[j];
                        if (n == 0 && a.auto_start) v = (r != 0.0) ? a.astart[coq + k] * q + a.half_T2 * fd : 0.0;
                        const double fe = a.fext ? (double)a.fext[(size_t)b * a.n_steps + n] * a.gain[(size_t)b * NQP + k] : 0.0;
                        v = a.kv[coq + k] * v - a.kq[coq + k] * q + r * (fe - fd);
                        q += v;
                        sq[j] = q; sv[j] = v;
#pragma unroll
                        for (int rep = 0; rep < FLOW_QREP; ++rep) st_tag(qx + (size_t)rep * NQP + k, (float)q, epoch);
                    }
                }
                if (a.timing && tid == 0) tkc = clock64();
                // ---- D: gather q^{n+1} ----
                // the last eight warps gather, 16 bytes per lane per load; the others go straight to the barrier
                if (warp >= NW - 8)
                    for (int pp = (warp - (NW - 8)) * 32 + lane; pp < NQP / 2; pp += 256)
                        *reinterpret_cast<float2 *>(q32 + 2 * pp) = ld_tag2(qx_mine + 2 * pp, epoch, s_abort);
            } else {
                bar_consumers(NC);
                for (int k = tid; k < NQP; k += NC) {
                    const double fd = (double)fpart[k], r = a.r[coq + k];
                    double q = sq[k], v = sv[k];
                    if (n == 0 && a.auto_start) v = (r != 0.0) ? a.astart[coq + k] * q + a.half_T2 * fd : 0.0;
                    const double fe = a.fext ? (double)a.fext[(size_t)b * a.n_steps + n] * a.gain[(size_t)b * NQP + k] : 0.0;
                    v = a.kv[coq + k] * v - a.kq[coq + k] * q + r * (fe - fd);
                    q += v;
                    sq[k] = q; sv[k] = v;
                    q32[k] = (float)q;
                }
            }
            bar_consumers(NC);
            if (a.timing && tid == 0) {
                const long long tk3 = clock64();
                long long *tm = a.timing + (size_t)blockIdx.x * 8;
                tm[0] += tk1 - tk0; tm[1] += tk2 - tk1; tm[2] += tk3 - tk2; tm[3] += tk3 - tk0;
                tm[4] += tkb - tk2; tm[5] += tkc - tkb; tm[6] += tk3 - tkc;
            }
        }
        if (out_cta && warp == NW - 1) {
            const int rem = a.n_steps & 31;
            if (rem && lane < rem) out[a.n_steps - rem + lane] = oreg;
            if (lane == 0) a.first_bad[b] = bad;
        }
        bar_consumers(NC);
    }
    if (tid == 0 && *s_abort) *a.timeout_flag = 1;
}

}  // namespace modal_dev
