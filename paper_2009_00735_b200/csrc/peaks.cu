// peaks.cu -- microbenchmarks for the roofline denominators of the on-chip kernels (include/aptsig_peaks.h).
//
// MEASURED_PEAKS.json carries HBM bandwidth and bf16 tensor throughput only; the signature kernels are bounded by
// plain FP32 issue, shared-memory atomics and shared-memory loads (project-and-bin = FMUL + 2 FFMA + FADD.RM
// + 1 shared atomic per (ion, direction) pair).  Each test runs one CTA of 1024 threads per SM (all resident at once),
// every warp issuing the same instruction `iters * kUnroll` times with independent operands, and is timed twice:
// CUDA events around the launch (rate per second) and clock64() inside every CTA (rate per SM clock; median CTA).
#include <algorithm>
#include <cstdint>
#include <vector>
#include <cuda_runtime.h>
#include "../../include/aptsig_peaks.h"

namespace {

constexpr int kThreads = 1024;
constexpr int kUnroll = 16;
constexpr int kSmemWords = 12288;          // 48 KB of shared memory: 384 rows of 32 banks

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int TEST>
__global__ void __launch_bounds__(kThreads, 1) k_peak(int iters, float seed, int zero, float *sink, long long *cycles)
{
    __shared__ __align__(16) uint32_t sm[kSmemWords];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < kSmemWords; i += kThreads) sm[i] = (uint32_t)i;
    __syncthreads();
    const uint32_t base = smem_addr(sm);
    float acc = 0.f;
    long long t0 = clock64();
    if (TEST == APX_PEAK_FFMA) {
        float a[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) a[u] = seed + (float)(u + lane);
        const float m = 1.0f + seed * 1e-9f, c = seed * 1e-7f;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) a[u] = __fmaf_rn(a[u], m, c);
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) acc += a[u];
    } else if (TEST == APX_PEAK_FFMA2) {
        uint64_t a[kUnroll];
        uint64_t m, c;
        {
            const float mf = 1.0f + seed * 1e-9f, cf = seed * 1e-7f;
            asm("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(mf));
            asm("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(cf));
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const float f = seed + (float)(u + lane);
            asm("mov.b64 %0, {%1, %1};" : "=l"(a[u]) : "f"(f));
        }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[u]) : "l"(m), "l"(c));
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            float lo, hi;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a[u]));
            acc += lo + hi;
        }
    } else if ((TEST >= APX_PEAK_RED_CONFLICT_FREE && TEST <= APX_PEAK_RED_RANDOM_BANK) || TEST == APX_PEAK_RED_INC_CONFLICT_FREE ||
               TEST == APX_PEAK_RED_SCATTERED_CONFLICT_FREE || TEST == APX_PEAK_RED_SCATTERED_HALVES) {
        // shared-memory reduction atomics without return value (the binning instruction); every warp works on its own
        // 12 rows of 32 words so that warps never share an address
        // increment from a kernel argument -> ATOMS.ADD (the high-u16 counters' 65536); the literal 1 of the INC test
        // compiles to ATOMS.POPC.INC (the low-u16 counters' form)
        const uint32_t inc = (uint32_t)seed;
        uint32_t lcg = (uint32_t)(tid * 2654435761u) | 1u;
        const uint32_t wbase = base + (uint32_t)warp * 12u * 128u;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                uint32_t off;
                const uint32_t row = (uint32_t)(u % 6);
                if (TEST == APX_PEAK_RED_CONFLICT_FREE || TEST == APX_PEAK_RED_INC_CONFLICT_FREE) off = row * 128u + (uint32_t)lane * 4u;   // 32 banks
                else if (TEST == APX_PEAK_RED_2WAY) off = (2u * row + (uint32_t)(lane >> 4)) * 128u + (uint32_t)(lane & 15) * 4u;
                else if (TEST == APX_PEAK_RED_SAME_ADDRESS) off = row * 128u;
                // 32 different banks, but every lane in a different 128-byte row (the binning pattern: a lane's row is its bin)
                else if (TEST == APX_PEAK_RED_SCATTERED_CONFLICT_FREE) off = (((uint32_t)lane * 5u + (uint32_t)u) % 12u) * 128u + (uint32_t)lane * 4u;
                // the kernel's layout: lanes 0-15 on the 16 banks {0-3, 8-11, 16-19, 24-27}, lanes 16-31 on the other 16, rows scattered
                else if (TEST == APX_PEAK_RED_SCATTERED_HALVES)
                    off = (((uint32_t)lane * 5u + (uint32_t)u) % 12u) * 128u + ((uint32_t)(lane & 3) + 8u * (uint32_t)((lane >> 2) & 3) + 4u * (uint32_t)(lane >> 4)) * 4u;
                else { lcg = lcg * 1664525u + 1013904223u; off = ((lcg >> 10) % (12u * 32u)) * 4u; }            // random word
                if (TEST == APX_PEAK_RED_INC_CONFLICT_FREE) asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(wbase + off) : "memory");
                else asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(wbase + off), "r"(inc) : "memory");
            }
        }
    } else {
        // shared-memory loads; results are folded into acc so that every load is live
        // (loads may reach into the rows of the following warps: wrap the warp's base so that everything stays inside sm[])
        // `zero` is a kernel argument that is 0 at run time: making the address formally depend on the iteration keeps the
        // compiler from hoisting the (loop-invariant) loads out of the timed loop
        const uint32_t wbase0 = base + (uint32_t)(warp % 26) * 12u * 128u;
        for (int it = 0; it < iters; ++it) {
            const uint32_t wbase = wbase0 + (uint32_t)(it * zero);
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                // sixteen DIFFERENT addresses per loop body: identical asm statements would be merged by the compiler
                if (TEST == APX_PEAK_LDS32_BROADCAST || TEST == APX_PEAK_LDS32_CONFLICT_FREE) {
                    const uint32_t off = TEST == APX_PEAK_LDS32_BROADCAST ? (uint32_t)u * 4u : (uint32_t)(u % 12) * 128u + (uint32_t)lane * 4u + (uint32_t)(u / 12) * 1536u;
                    float v;
                    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(wbase + off) : "memory");
                    acc += v;
                } else {
                    uint32_t off;
                    const uint32_t row = (uint32_t)u * 64u;                                              // 16 rows of 64 B
                    if (TEST == APX_PEAK_LDS128_BROADCAST_1) off = row;                                   // one address per warp
                    else if (TEST == APX_PEAK_LDS128_BROADCAST_2) off = row + (uint32_t)(lane >> 4) * 16u;     // two (half-warps)
                    else if (TEST == APX_PEAK_LDS128_BROADCAST_4) off = row + (uint32_t)(lane >> 3) * 16u;     // four (quarter-warps)
                    else off = (uint32_t)(u % 3) * 512u + (uint32_t)lane * 16u + (uint32_t)(u / 3) * 1536u;    // 512 B per instruction
                    float x, y, z, w;
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x), "=f"(y), "=f"(z), "=f"(w) : "r"(wbase + off) : "memory");
                    acc += x + y + z + w;
                }
            }
        }
    }
    long long t1 = clock64();
    __syncthreads();
    if (tid == 0) cycles[blockIdx.x] = t1 - t0;
    if (acc == 123.456f) sink[0] = acc + (float)sm[lane];      // keeps the arithmetic and the atomics' target alive
}

template <int TEST>
cudaError_t run_test(int blocks, int iters, float *sink, long long *cycles, float *ms)
{
    cudaEvent_t a, b;
    cudaError_t e = cudaEventCreate(&a);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&b);
    if (e != cudaSuccess) return e;
    k_peak<TEST><<<blocks, kThreads>>>(iters / 8 + 1, 1.0f, 0, sink, cycles);      // warm-up
    cudaEventRecord(a);
    k_peak<TEST><<<blocks, kThreads>>>(iters, 1.0f, 0, sink, cycles);
    cudaEventRecord(b);
    e = cudaEventSynchronize(b);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, a, b);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return e;
}

}  // namespace

extern "C" const char *apx_peak_name(int test)
{
    switch (test) {
        case APX_PEAK_FFMA: return "ffma";
        case APX_PEAK_FFMA2: return "ffma2_packed";
        case APX_PEAK_RED_CONFLICT_FREE: return "red_shared_conflict_free";
        case APX_PEAK_RED_2WAY: return "red_shared_2way_conflict";
        case APX_PEAK_RED_SAME_ADDRESS: return "red_shared_same_address";
        case APX_PEAK_RED_RANDOM_BANK: return "red_shared_random_word";
        case APX_PEAK_LDS32_BROADCAST: return "lds32_broadcast";
        case APX_PEAK_LDS32_CONFLICT_FREE: return "lds32_conflict_free";
        case APX_PEAK_LDS128_BROADCAST_1: return "lds128_broadcast_1_address";
        case APX_PEAK_LDS128_BROADCAST_2: return "lds128_broadcast_2_addresses";
        case APX_PEAK_LDS128_BROADCAST_4: return "lds128_broadcast_4_addresses";
        case APX_PEAK_LDS128_CONFLICT_FREE: return "lds128_conflict_free";
        case APX_PEAK_RED_INC_CONFLICT_FREE: return "red_shared_inc_conflict_free";
        case APX_PEAK_RED_SCATTERED_CONFLICT_FREE: return "red_shared_scattered_rows_conflict_free";
        case APX_PEAK_RED_SCATTERED_HALVES: return "red_shared_scattered_rows_half_warp_banks";
        default: return nullptr;
    }
}

extern "C" int apx_peak_measure(int device, int test, int iters, apx_peak_result *out)
{
    if (!out || iters < 1 || !apx_peak_name(test)) return -1;
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return -3;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return -3;
    const int blocks = prop.multiProcessorCount;
    float *sink = nullptr;
    long long *cycles = nullptr;
    cudaError_t e = cudaMalloc(&sink, 4);
    if (e == cudaSuccess) e = cudaMalloc(&cycles, sizeof(long long) * blocks);
    float ms = 0.f;
    if (e == cudaSuccess) {
        switch (test) {
#define CASE(T) case T: e = run_test<T>(blocks, iters, sink, cycles, &ms); break;
            CASE(APX_PEAK_FFMA) CASE(APX_PEAK_FFMA2) CASE(APX_PEAK_RED_CONFLICT_FREE) CASE(APX_PEAK_RED_2WAY)
            CASE(APX_PEAK_RED_SAME_ADDRESS) CASE(APX_PEAK_RED_RANDOM_BANK) CASE(APX_PEAK_LDS32_BROADCAST)
            CASE(APX_PEAK_LDS32_CONFLICT_FREE) CASE(APX_PEAK_LDS128_BROADCAST_1) CASE(APX_PEAK_LDS128_BROADCAST_2)
            CASE(APX_PEAK_LDS128_BROADCAST_4) CASE(APX_PEAK_LDS128_CONFLICT_FREE) CASE(APX_PEAK_RED_INC_CONFLICT_FREE) CASE(APX_PEAK_RED_SCATTERED_CONFLICT_FREE)
            CASE(APX_PEAK_RED_SCATTERED_HALVES)
#undef CASE
        }
    }
    std::vector<long long> cyc(blocks, 0);
    if (e == cudaSuccess) e = cudaMemcpy(cyc.data(), cycles, sizeof(long long) * blocks, cudaMemcpyDeviceToHost);
    if (sink) cudaFree(sink);
    if (cycles) cudaFree(cycles);
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    if (e != cudaSuccess) return -3;
    std::sort(cyc.begin(), cyc.end());
    const double warp_inst_per_cta = (double)(kThreads / 32) * (double)iters * kUnroll;
    out->sm_count = blocks;
    out->ms = ms;
    out->median_cycles = (double)cyc[blocks / 2];
    out->warp_inst_per_s = warp_inst_per_cta * blocks / (ms * 1e-3);
    out->warp_inst_per_clk_per_sm = warp_inst_per_cta / out->median_cycles;
    out->sm_mhz_effective = out->median_cycles / (ms * 1e-3) / 1e6;
    return 0;
}
