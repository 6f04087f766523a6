// vk_static.cu -- modal_vk_simulate_static: the von Karman recurrence through ONE entry point that allocates nothing.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it): every
// input and output is a DEVICE pointer of the caller, and the cross-CTA exchange buffer -- the only scratch memory the kernel
// needs -- is a file-scope static __device__ array of MODAL_STATIC_SCRATCH_BYTES that every GPU which loads the library holds
// until the process exits.  No plan, no cudaMalloc / cudaFree, no allocating library routine, no host synchronisation.
//
// The kernel is a variant of vk_flow_kernel (vk_flow.cuh): a team of G CTAs per sample, the in-plane modes n split over the team,
// the partial forces exchanged one-way through L2 as tagged 64-bit words {fp32 value, step epoch} (st_tag / ld_tag of vk_flow.cuh)
// and summed by every CTA in team order, so the team's CTAs hold bit-identical replicas of the fp64 state.  Per step
// (Eq. 9-11 with C eliminated; recurrence PAPER.md:153-161 Eq. 19/20 in delta form, R4):
//   t_n[k] = sum_r H^n[k][r] q[r];  G_n = sum_k q[k] t_n[k];  eta_n = s_n G_n;  f[k] = sum_n eta_n t_n[k]          (fp32)
//   v <- -c2 v - (1 - c1 - c2) q - c3 f;  q <- q + v   ( == q^{n+1} = c1 q^n + c2 q^{n-1} - c3 f )                     (fp64)
//   out[b][n] = sum_k w[k] q^n[k]
// H is read dense from global memory (L2) every step, as uploaded: this entry point trades the packed, parity-skipping layouts
// of the plan-based kernels for having no set-up that allocates.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstring>
#include <mutex>
#include "../../include/modal.h"
#include "vk_flow.cuh"   // st_tag / ld_tag (bounded waits), FLOW_FULL

namespace md = modal_dev;

namespace {

// The scratch: [step parity][sample of the launch][team member][n_q] tagged words.  In host code this name is only a stand-in
// for the symbol -- the device address comes from cudaGetSymbolAddress (static_setup below); device code may name it directly.
static __device__ __align__(256) unsigned char modal_static_scratch[MODAL_STATIC_SCRATCH_BYTES];

constexpr int ST_THREADS_S = 256;      // one thread per transverse mode (n_q <= MODAL_STATIC_MAX_NQ == 256), 8 warps
constexpr int ST_G_MAX = 16;           // most CTAs of a team

struct StaticArgs {
    int n_q, n_phi, batch, n_steps, G, cb_q, cb_phi;      // cb_*: coefficient row stride per sample (0: one row for all)
    const float *H; const double *c1, *c2, *c3; const float *s, *w;
    const double *q0, *qm1;
    float *out; int *first_bad;
    unsigned long long *scratch;                          // device address of modal_static_scratch
};

// sums of a and b over the block, in a fixed order; every thread gets both.  red: 16 floats.  Two barriers.
__device__ __forceinline__ void block_sum2(float a, float b, float *red, float &A, float &B)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) { a += __shfl_xor_sync(md::FLOW_FULL, a, m); b += __shfl_xor_sync(md::FLOW_FULL, b, m); }
    if (lane == 0) { red[warp] = a; red[8 + warp] = b; }
    __syncthreads();
    A = ((red[0] + red[1]) + (red[2] + red[3])) + ((red[4] + red[5]) + (red[6] + red[7]));
    B = ((red[8] + red[9]) + (red[10] + red[11])) + ((red[12] + red[13]) + (red[14] + red[15]));
    __syncthreads();
}

__global__ void __launch_bounds__(ST_THREADS_S) vk_static_kernel(const StaticArgs a)
{
    __shared__ float qf[MODAL_STATIC_MAX_NQ], tn[MODAL_STATIC_MAX_NQ], red[16];
    __shared__ volatile int s_abort;
    const int k = threadIdx.x, lane = k & 31, warp = k >> 5;
    const int bl = blockIdx.x / a.G, g = blockIdx.x - bl * a.G;           // sample of this launch, team member
    const int n0 = (int)((long long)a.n_phi * g / a.G), n1 = (int)((long long)a.n_phi * (g + 1) / a.G);
    const bool mine = k < a.n_q;
    const size_t cq = (size_t)bl * a.cb_q, cp = (size_t)bl * a.cb_phi;
    double q = 0.0, v = 0.0, kv = 0.0, kq = 0.0, r = 0.0; float wk = 0.f;
    if (mine) {
        q = a.q0[(size_t)bl * a.n_q + k]; v = q - a.qm1[(size_t)bl * a.n_q + k];
        const double c1 = a.c1[cq + k], c2 = a.c2[cq + k];
        kv = -c2; kq = 1.0 - c1 - c2; r = a.c3[cq + k]; wk = a.w[cq + k];
    }
    if (k == 0) s_abort = 0;
    int sbad = -1;
    const float *s = a.s + cp;
    for (int n = 0; n < a.n_steps; ++n) {
        const float x = (float)q;
        qf[k] = x;                                  // k >= n_q: zero
        __syncthreads();
        float o, nr;
        block_sum2(wk * x, x * x, red, o, nr);      // a1 pickup + a6 write-out, and the non-finite check
        if (g == 0 && k == 0) {
            a.out[(size_t)bl * a.n_steps + n] = o;
            if (sbad < 0 && !(isfinite(o) && isfinite(nr))) sbad = n;
        }
        float facc = 0.f;
        for (int nn = n0; nn < n1; ++nn) {
            const float *Hn = a.H + (size_t)nn * a.n_q * a.n_q;
            for (int row = warp; row < a.n_q; row += 8) {                 // a2: one warp per row of H^n, coalesced
                const float *hr = Hn + (size_t)row * a.n_q;
                float p = 0.f;
                for (int c = lane; c < a.n_q; c += 32) p = fmaf(__ldg(hr + c), qf[c], p);
#pragma unroll
                for (int m = 16; m >= 1; m >>= 1) p += __shfl_xor_sync(md::FLOW_FULL, p, m);
                if (lane == 0) tn[row] = p;
            }
            __syncthreads();
            const float t = mine ? tn[k] : 0.f;
            float Gn, unused;
            block_sum2(x * t, 0.f, red, Gn, unused);                      // a3 (the second barrier also protects tn)
            facc = fmaf(s[nn] * Gn, t, facc);                             // a4
        }
        float f = facc;
        if (a.G > 1) {                                                    // team exchange through the static scratch
            unsigned long long *base = a.scratch + (((size_t)(n & 1) * a.batch + bl) * a.G) * MODAL_STATIC_MAX_NQ;
            if (mine) {
                md::st_tag(base + (size_t)g * MODAL_STATIC_MAX_NQ + k, facc, (unsigned)n + 1u);
                // all G loads in flight together (one after the other they cost an L2 round trip each); summed in team order:
                // identical bits in every CTA of the team
                float vv[ST_G_MAX];
                unsigned pend = (1u << a.G) - 1u, spins = 0;
                while (pend) {
                    unsigned long long w0[ST_G_MAX];
#pragma unroll
                    for (int gg = 0; gg < ST_G_MAX; ++gg)
                        if (pend >> gg & 1)
                            asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(w0[gg]) : "l"(base + (size_t)gg * MODAL_STATIC_MAX_NQ + k) : "memory");
#pragma unroll
                    for (int gg = 0; gg < ST_G_MAX; ++gg)
                        if ((pend >> gg & 1) && (unsigned)(w0[gg] >> 32) == (unsigned)n + 1u) { vv[gg] = __uint_as_float((unsigned)w0[gg]); pend &= ~(1u << gg); }
                    if (pend && (++spins & 1023u) == 0 && (s_abort || spins > (1u << 21))) { s_abort = 1; break; }
                }
                f = 0.f;
#pragma unroll
                for (int gg = 0; gg < ST_G_MAX; ++gg) if (gg < a.G) f += vv[gg];
            }
        }
        v = fma(kv, v, fma(-kq, q, -r * (double)f));                      // a5
        q += v;
        __syncthreads();                                                  // qf is rewritten at the top
    }
    if (k == 0 && a.first_bad) {
        if (s_abort) atomicMin(a.first_bad + bl, -2);                     // an exchange timed out (team not co-resident)
        else if (g == 0 && sbad >= 0) atomicCAS(a.first_bad + bl, -1, sbad);
    }
}

struct DeviceSetup { bool done = false; unsigned long long *scratch = nullptr; int sm = 0; };
DeviceSetup g_setup[64];
std::mutex g_mutex;

void say(char *err, int err_bytes, const char *msg)
{
    if (err && err_bytes > 0) snprintf(err, (size_t)err_bytes, "%s", msg);
}

// once per device, with that device current: the device address of the scratch symbol and the SM count
cudaError_t static_setup(int dev, DeviceSetup **out)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    DeviceSetup &d = g_setup[dev];
    if (!d.done) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, modal_static_scratch);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&d.sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        d.scratch = static_cast<unsigned long long *>(p);
        d.done = true;
    }
    *out = &d;
    return cudaSuccess;
}

}  // namespace

extern "C" modal_status modal_vk_simulate_static(int n_q, int n_phi, int batch, int n_steps, int coeff_batch,
                                                 const float *H_dev, const double *c1_dev, const double *c2_dev, const double *c3_dev,
                                                 const float *s_dev, const float *w_dev, const double *q0_dev, const double *qm1_dev,
                                                 float *out_audio_dev, int *first_bad_dev, void *cuda_stream, char *err, int err_bytes)
{
    char buf[256];
    if (err && err_bytes > 0) err[0] = 0;
    if (n_q < 1 || n_phi < 1 || batch < 0 || n_steps < 0 || (coeff_batch != 1 && coeff_batch != batch && batch > 0)) {
        say(err, err_bytes, "modal_vk_simulate_static: n_q, n_phi >= 1, batch, n_steps >= 0 and coeff_batch in {1, batch} are required");
        return MODAL_EINVAL;
    }
    if (n_q > MODAL_STATIC_MAX_NQ) {
        snprintf(buf, sizeof buf, "modal_vk_simulate_static: n_q = %d exceeds MODAL_STATIC_MAX_NQ = %d (use a plan and modal_simulate)", n_q, MODAL_STATIC_MAX_NQ);
        say(err, err_bytes, buf);
        return MODAL_EINCOMPAT;
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    DeviceSetup *ds = nullptr;
    if (e == cudaSuccess && (dev < 0 || dev >= 64)) { say(err, err_bytes, "modal_vk_simulate_static: device ordinal beyond 63"); return MODAL_EINCOMPAT; }
    if (e == cudaSuccess) e = static_setup(dev, &ds);
    if (e != cudaSuccess) {
        snprintf(buf, sizeof buf, "modal_vk_simulate_static: CUDA set-up failed: %s", cudaGetErrorString(e));
        say(err, err_bytes, buf); cudaGetLastError();
        return MODAL_ECUDA;
    }
    if (batch == 0 || n_steps == 0) return MODAL_OK;                      // set-up only (e.g. once before a graph capture)
    if (!H_dev || !c1_dev || !c2_dev || !c3_dev || !s_dev || !w_dev || !q0_dev || !qm1_dev || !out_audio_dev) {
        say(err, err_bytes, "modal_vk_simulate_static: a required device pointer is NULL (only first_bad_dev, err may be)");
        return MODAL_EINVAL;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // samples per launch and CTAs per team: every CTA of a launch must be co-resident (one per SM), and the launch's exchange
    // words [2][samples][G][MODAL_STATIC_MAX_NQ] x 8 B must fit the static array
    const int per_launch = batch < ds->sm ? batch : ds->sm;
    int G = ds->sm / per_launch;
    if (G > n_phi) G = n_phi;
    if (G > ST_G_MAX) G = ST_G_MAX;
    while (G > 1 && (size_t)2 * per_launch * G * MODAL_STATIC_MAX_NQ * 8 > MODAL_STATIC_SCRATCH_BYTES) --G;
    const size_t need = G > 1 ? (size_t)2 * per_launch * G * MODAL_STATIC_MAX_NQ * 8 : 0;
    if (need > MODAL_STATIC_SCRATCH_BYTES) {       // cannot happen with the limits above; kept as the guard the array's size demands
        snprintf(buf, sizeof buf, "modal_vk_simulate_static: %zu bytes of exchange scratch exceed MODAL_STATIC_SCRATCH_BYTES = %u", need, (unsigned)MODAL_STATIC_SCRATCH_BYTES);
        say(err, err_bytes, buf);
        return MODAL_EINCOMPAT;
    }
    if (first_bad_dev) { e = cudaMemsetAsync(first_bad_dev, 0xff, (size_t)batch * sizeof(int), st); if (e != cudaSuccess) goto fail; }
    for (int b0 = 0; b0 < batch; b0 += per_launch) {
        const int nb = batch - b0 < per_launch ? batch - b0 : per_launch;
        StaticArgs a{};
        a.n_q = n_q; a.n_phi = n_phi; a.batch = nb; a.n_steps = n_steps; a.G = G;
        a.cb_q = coeff_batch == 1 ? 0 : n_q; a.cb_phi = coeff_batch == 1 ? 0 : n_phi;
        const size_t oq = coeff_batch == 1 ? 0 : (size_t)b0 * n_q, op = coeff_batch == 1 ? 0 : (size_t)b0 * n_phi;
        a.H = H_dev; a.c1 = c1_dev + oq; a.c2 = c2_dev + oq; a.c3 = c3_dev + oq; a.s = s_dev + op; a.w = w_dev + oq;
        a.q0 = q0_dev + (size_t)b0 * n_q; a.qm1 = qm1_dev + (size_t)b0 * n_q;
        a.out = out_audio_dev + (size_t)b0 * n_steps; a.first_bad = first_bad_dev ? first_bad_dev + b0 : nullptr;
        a.scratch = ds->scratch;
        // the array keeps the last call's words, whose epochs would match this call's: clear what this launch reads
        if (G > 1) { e = cudaMemsetAsync(ds->scratch, 0, (size_t)2 * nb * G * MODAL_STATIC_MAX_NQ * 8, st); if (e != cudaSuccess) goto fail; }
        vk_static_kernel<<<nb * G, ST_THREADS_S, 0, st>>>(a);
        e = cudaGetLastError();
        if (e != cudaSuccess) goto fail;
    }
    return MODAL_OK;
fail:
    snprintf(buf, sizeof buf, "modal_vk_simulate_static: %s", cudaGetErrorString(e));
    say(err, err_bytes, buf); cudaGetLastError();
    return MODAL_ECUDA;
}
