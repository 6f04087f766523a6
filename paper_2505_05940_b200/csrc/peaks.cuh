// peaks.cuh -- micro-kernels behind modal_measure_peaks(): the denominators the roofline fractions of this build are
// quoted against that MEASURED_PEAKS.json does not hold ("FP32-pipe, SMEM and L2 peaks ... the builder must
// measure them"), plus the latency of the cross-CTA exchange primitives the persistent kernels are built on.
//   fma_peak<T>      FP32 / FP64 FMA issue peak (8 independent chains per thread, all SMs, 8 CTAs of 256 threads per SM)
//   read_sweep       ld.global.cg.v4 sweep of a buffer, repeated: 8 MiB and 64 MiB working sets stay in the 126 MB L2,
//                    1 GiB streams from HBM
//   smem_read        conflict-free LDS.128 of a 64 KiB shared-memory block by 512 threads
//   tmem_read        tcgen05.ld.32x32b.x32 of a 512-column TMEM allocation by four warps (the epilogue pattern of vk_mma)
//   hop              ping-pong of one tagged 8-byte word between CTA 0 and CTA 1 (st.relaxed.gpu / polling ld.relaxed.gpu),
//                    and the same with release / acquire on a flag next to a payload line; optionally while the other 146
//                    CTAs keep the L2 busy with a read sweep ("under load")
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace modal_dev {

template <class T>
__global__ void __launch_bounds__(256) peak_fma_kernel(T *out, int iters, T x0)
{
    T a0 = x0 + (T)threadIdx.x, a1 = a0 + (T)1, a2 = a0 + (T)2, a3 = a0 + (T)3, a4 = a0 + (T)4, a5 = a0 + (T)5, a6 = a0 + (T)6, a7 = a0 + (T)7;
    const T m = (T)0.999999, c = (T)1e-7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = a0 * m + c; a1 = a1 * m + c; a2 = a2 * m + c; a3 = a3 * m + c;
            a4 = a4 * m + c; a5 = a5 * m + c; a6 = a6 * m + c; a7 = a7 * m + c;
        }
    }
    const T s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s == (T)-1) out[blockIdx.x * blockDim.x + threadIdx.x] = s;       // never true: keeps the chains alive
}

__global__ void __launch_bounds__(512) peak_read_sweep_kernel(const uint4 *buf, size_t n16, int passes, unsigned *sink)
{
    unsigned acc = 0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; ++p)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += 4 * stride) {
            uint4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) v[u] = i + u * stride < n16 ? __ldcg(buf + i + u * stride) : make_uint4(0, 0, 0, 0);
#pragma unroll
            for (int u = 0; u < 4; ++u) acc += v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
        }
    if (acc == 0x12345678u) *sink = acc;
}

__global__ void __launch_bounds__(512) peak_smem_read_kernel(int iters, long long *cycles, unsigned *sink)
{
    extern __shared__ __align__(16) unsigned char peak_smem[];
    uint4 *s = reinterpret_cast<uint4 *>(peak_smem);
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) s[i] = make_uint4(0, 0, 0, 0);      // zeros: acc stays 0, rot = it * 32
    __syncthreads();
    unsigned acc = 0;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        const int rot = (it * 32 + (int)acc) & 4095;        // data-dependent rotation: the loads cannot be hoisted out of the loop
#pragma unroll
        for (int u = 0; u < 8; ++u) {                       // 8 x 512 threads x 16 B = 64 KiB per iteration, lane-contiguous
            const uint4 v = s[(u * 512 + threadIdx.x + rot) & 4095];
            acc += v.x ^ v.y ^ v.z ^ v.w;
        }
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
    if (acc == 0x12345678u) *sink = acc;
}

__global__ void __launch_bounds__(128) peak_tmem_read_kernel(int iters, long long *cycles, unsigned *sink)
{
    __shared__ uint32_t tptr;
    const int warp = threadIdx.x >> 5;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&tptr)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t base = tptr + ((uint32_t)(warp * 32) << 16);
    unsigned acc = 0;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it)
        for (int c = 0; c < 512; c += 64) {                 // two x32 loads in flight per wait
            uint32_t v[64];
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                         "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                         : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                           "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
                           "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
                           "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31]) : "r"(base + c));
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                         "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                         : "=r"(v[32]), "=r"(v[33]), "=r"(v[34]), "=r"(v[35]), "=r"(v[36]), "=r"(v[37]), "=r"(v[38]), "=r"(v[39]), "=r"(v[40]),
                           "=r"(v[41]), "=r"(v[42]), "=r"(v[43]), "=r"(v[44]), "=r"(v[45]), "=r"(v[46]), "=r"(v[47]), "=r"(v[48]), "=r"(v[49]),
                           "=r"(v[50]), "=r"(v[51]), "=r"(v[52]), "=r"(v[53]), "=r"(v[54]), "=r"(v[55]), "=r"(v[56]), "=r"(v[57]), "=r"(v[58]),
                           "=r"(v[59]), "=r"(v[60]), "=r"(v[61]), "=r"(v[62]), "=r"(v[63]) : "r"(base + c + 32));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int u = 0; u < 64; u += 8) acc += v[u];
        }
    const long long t1 = clock64();
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
    if (acc == 0x12345678u) *sink = acc;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tptr), "r"(512));
}

// CTA 0 and CTA 1: `rounds` round trips of a word.  mode 0: the word itself is polled (st.relaxed.gpu / ld.relaxed.gpu, the
// tagged-word hops of vk_flow / vk_mma); mode 1: a 128-byte payload is written, then a flag with st.release.gpu, the reader
// polls the flag (relaxed), reads it once with ld.acquire.gpu and then the payload (the q hop of vk_mma).  The other CTAs
// sweep `bg` (L2 resident) until CTA 0 raises *stop, when `load` is set.  cycles[0] = cycles of CTA 0 for all rounds.
__global__ void __launch_bounds__(512) peak_hop_kernel(unsigned long long *words, unsigned *payload, int rounds, int mode, int load,
                                                       const uint4 *bg, size_t bg16, volatile int *stop, long long *cycles, unsigned *sink)
{
    if (blockIdx.x >= 2) {
        if (!load) return;
        unsigned acc = 0;
        for (int guard = 0; !*stop && guard < (1 << 20); ++guard)
            for (size_t i = (size_t)(blockIdx.x - 2) * blockDim.x + threadIdx.x; i < bg16; i += (size_t)8 * (gridDim.x - 2) * blockDim.x) {
                uint4 v[8];                                  // eight 16-byte loads in flight per thread: the sweep runs near the L2 read peak
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const size_t x = i + (size_t)u * (gridDim.x - 2) * blockDim.x;
                    v[u] = x < bg16 ? __ldcg(bg + x) : make_uint4(0, 0, 0, 0);
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) acc += v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
            }
        if (acc == 0x12345678u) *sink = acc;
        return;
    }
    if (threadIdx.x != 0) return;
    const int me = blockIdx.x;
    unsigned long long *mine = words + me * 32, *theirs = words + (1 - me) * 32;       // 256 bytes apart
    unsigned *pm = payload + me * 64, *pt = payload + (1 - me) * 64;
    unsigned acc = 0;
    const long long t0 = clock64();
    bool dead = false;
    for (int r = 1; r <= rounds && !dead; ++r) {
        unsigned long long w;
        unsigned spins = 0;
        if (me == 1) {                                       // CTA 1 answers: wait for round r of CTA 0 first
            do { asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(w) : "l"(theirs) : "memory"); } while ((unsigned)(w >> 32) != (unsigned)r && ++spins < (1u << 24));
            if (mode == 1) {
                asm volatile("ld.acquire.gpu.global.b64 %0, [%1];" : "=l"(w) : "l"(theirs) : "memory");
                acc += __ldcg(pt + (r & 31));
            }
        }
        if (mode == 1) { pm[r & 31] = (unsigned)r; asm volatile("st.release.gpu.global.b64 [%0], %1;" ::"l"(mine), "l"(((unsigned long long)r << 32) | 1ull) : "memory"); }
        else asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(mine), "l"(((unsigned long long)r << 32) | 1ull) : "memory");
        if (me == 0) {                                       // CTA 0 waits for the answer of round r
            do { asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(w) : "l"(theirs) : "memory"); } while ((unsigned)(w >> 32) != (unsigned)r && ++spins < (1u << 24));
            if (mode == 1) {
                asm volatile("ld.acquire.gpu.global.b64 %0, [%1];" : "=l"(w) : "l"(theirs) : "memory");
                acc += __ldcg(pt + (r & 31));
            }
        }
        dead = spins >= (1u << 24);                          // bounded: a partner that never runs ends the measurement, not the GPU
    }
    const long long t1 = clock64();
    if (me == 0) { cycles[0] = dead ? -1 : t1 - t0; *stop = 1; __threadfence(); }
    if (acc == 0x12345678u) *sink = acc;
}

}  // namespace modal_dev
