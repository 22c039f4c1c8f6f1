// fsp.cu -- reciprocal space method (Eq. 2; cost L389-393: N_roi x N_w x L_D^3).
//
//   F(k) = sum_w exp(-2 pi i k.(p_w - p_c)),  k on an L^3 grid over [-k_max, k_max]^3, signature = |F| (reading #25).
//
// The phase factorises per axis, exp(-2 pi i k.d) = ex_w[ix] ey_w[iy] ez_w[iz], so one z-slice of the image is the complex
// contraction  C[iy][ix] = sum_w (ez_w[iz] ey_w[iy]) * ex_w[ix]  =  A[iy][w] . E[w][ix]  with K = N_w: a dense complex GEMM
// per (material point, iz).  This version runs it on the FP32 pipe, SGEMM style: CTA = (material point, iz, 64 x 64 tile of
// (iy, ix)), 256 threads with a 4 x 4 complex register tile each, ions in steps of 32 whose phase factors are built in
// shared memory with sincospif (exact argument reduction in units of pi).  The ROI gather (cell rows of the plan's
// sorted cloud, exact fp32 ball test) is the one of the signature kernels.  ROIs with more ions than the shared buffer
// are handled by streaming the candidate ions of their cell rows through the same loop with non-members masked to zero.
#include <cmath>
#include <mutex>
#include "common.cuh"
#include "../../include/aptsig_ext.h"

namespace apx {

constexpr int kFspThreads = 256;
constexpr int kFspTile = 64;             // (iy, ix) tile edge
constexpr int kFspStep = 32;             // ions per K step
constexpr int kFspCap = 6144;            // ions held in shared memory (72 KB); larger ROIs stream their candidates

struct FspParams {
    const float4 *sorted;
    const uint32_t *cell_start;
    const GridParams *grid;
    const float *centres;
    const float *kaxis;       // [L] k values of one axis, fp64 on the host rounded once to fp32
    float *out;               // [M][L][L][L] amplitude
    uint32_t *counts;
    const uint32_t *list;     // nullptr: every material point; else list[0] = count, list[1..] = the material points to serve
                              // (those the tensor-core kernel k_fsp_mma left out: more ions than its shared buffer)
    int L, tiles;             // tiles per axis = ceil(L / 64)
    float R, R2;
};

// phase factor exp(-2 pi i k d): sincospif takes the angle in units of pi, its argument reduction is exact
__device__ __forceinline__ float2 phase(float k, float d)
{
    float s, c;
    sincospif(-2.0f * __fmul_rn(k, d), &s, &c);
    return make_float2(c, s);
}

__global__ void __launch_bounds__(kFspThreads, 2) k_fsp(const FspParams p)
{
    extern __shared__ __align__(16) float fsm[];
    float *a_re = fsm;                                   // [kFspStep][64]  A[w][iy] = ez_w ey_w[iy]
    float *a_im = a_re + kFspStep * kFspTile;
    float *e_re = a_im + kFspStep * kFspTile;            // [kFspStep][64]  E[w][ix] = ex_w[ix]
    float *e_im = e_re + kFspStep * kFspTile;
    float *step_ion = e_im + kFspStep * kFspTile;        // [kFspStep][4]   dx, dy, dz, weight (1 = member, 0 = masked)
    float *ions = step_ion + kFspStep * 4;               // [kFspCap][3]
    __shared__ int s_n;

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int L = p.L;
    const GridParams g = *p.grid;
    const int64_t per_point = (int64_t)L * p.tiles * p.tiles;
    const int64_t n_items = p.list ? (int64_t)p.list[0] * per_point : (int64_t)gridDim.x;
  for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
    int64_t b = item;
    const int tx_tile = (int)(b % p.tiles); b /= p.tiles;
    const int ty_tile = (int)(b % p.tiles); b /= p.tiles;
    const int iz = (int)(b % L);
    const int64_t m = p.list ? (int64_t)p.list[1 + b / L] : b / L;
    __syncthreads();                                  // the previous item is done with the shared buffers
    const float cx = p.centres[3 * m], cy = p.centres[3 * m + 1], cz = p.centres[3 * m + 2];
    const RoiCells rc = roi_cells(g, cx, cy, cz, p.R);
    const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
    if (tid == 0) s_n = 0;
    __syncthreads();
    // ---- gather (step a2 of the signature path): members' d = p - c into shared memory, count in s_n -----------------
    if (g.n_accepted) {
        for (int row = wid; row < ny_r * nz_r; row += kFspThreads / 32) {
            const int iy = rc.iy0 + row % ny_r, izc = rc.iz0 + row / ny_r;
            const int base = (izc * g.ny + iy) * g.nx;
            const uint32_t beg = p.cell_start[base + rc.ix0], end = p.cell_start[base + rc.ix1 + 1];
            for (uint32_t i = beg + lane; i < ((end - beg + 31u) & ~31u) + beg; i += 32) {
                bool in = false;
                float dx = 0.f, dy = 0.f, dz = 0.f;
                if (i < end) {
                    const float4 q = p.sorted[i];
                    dx = __fsub_rn(q.x, cx); dy = __fsub_rn(q.y, cy); dz = __fsub_rn(q.z, cz);
                    in = inside(dx, dy, dz, p.R2);
                }
                const unsigned msk = __ballot_sync(0xffffffffu, in);
                if (msk) {
                    int pos = 0;
                    if (lane == 0) pos = atomicAdd(&s_n, __popc(msk));
                    pos = __shfl_sync(0xffffffffu, pos, 0) + __popc(msk & ((1u << lane) - 1u));
                    if (in && pos < kFspCap) { ions[3 * pos] = dx; ions[3 * pos + 1] = dy; ions[3 * pos + 2] = dz; }
                }
            }
        }
    }
    __syncthreads();
    const int n = s_n;
    if (p.counts && iz == 0 && tx_tile == 0 && ty_tile == 0 && tid == 0) p.counts[m] = (uint32_t)n;
    const bool streaming = n > kFspCap;

    const int ty = tid >> 4, tx = tid & 15;               // 16 x 16 threads, 4 x 4 complex outputs each
    const int iy0 = ty_tile * kFspTile, ix0 = tx_tile * kFspTile;
    const float kz = p.kaxis[iz];
    float cr[4][4], ci[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) { cr[i][j] = 0.f; ci[i][j] = 0.f; }

    // one K step over the kFspStep ions in step_ion: build A and E, then the register-tile update
    auto k_step = [&](int cnt) {
        __syncthreads();                                  // step_ion written; previous step's tiles consumed
        for (int e = tid; e < kFspStep * kFspTile; e += kFspThreads) {
            const int w = e >> 6, c = e & 63;
            float2 a = make_float2(0.f, 0.f), ex = make_float2(0.f, 0.f);
            if (w < cnt) {
                const float dx = step_ion[4 * w], dy = step_ion[4 * w + 1], dz = step_ion[4 * w + 2], wt = step_ion[4 * w + 3];
                if (wt != 0.f) {
                    if (iy0 + c < L) {
                        const float2 ez = phase(kz, dz), ey = phase(p.kaxis[iy0 + c], dy);
                        a = make_float2(ez.x * ey.x - ez.y * ey.y, ez.x * ey.y + ez.y * ey.x);
                    }
                    if (ix0 + c < L) ex = phase(p.kaxis[ix0 + c], dx);
                }
            }
            a_re[e] = a.x; a_im[e] = a.y; e_re[e] = ex.x; e_im[e] = ex.y;
        }
        __syncthreads();
#pragma unroll 4
        for (int w = 0; w < kFspStep; ++w) {
            const float4 ar = *reinterpret_cast<const float4 *>(a_re + w * kFspTile + 4 * ty);
            const float4 ai = *reinterpret_cast<const float4 *>(a_im + w * kFspTile + 4 * ty);
            const float4 er = *reinterpret_cast<const float4 *>(e_re + w * kFspTile + 4 * tx);
            const float4 ei = *reinterpret_cast<const float4 *>(e_im + w * kFspTile + 4 * tx);
            const float arr[4] = {ar.x, ar.y, ar.z, ar.w}, aii[4] = {ai.x, ai.y, ai.z, ai.w};
            const float err[4] = {er.x, er.y, er.z, er.w}, eii[4] = {ei.x, ei.y, ei.z, ei.w};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    cr[i][j] = fmaf(arr[i], err[j], cr[i][j]);
                    cr[i][j] = fmaf(-aii[i], eii[j], cr[i][j]);
                    ci[i][j] = fmaf(arr[i], eii[j], ci[i][j]);
                    ci[i][j] = fmaf(aii[i], err[j], ci[i][j]);
                }
        }
    };

    if (!streaming) {
        for (int w0 = 0; w0 < n; w0 += kFspStep) {
            const int cnt = min(kFspStep, n - w0);
            __syncthreads();                              // the previous step has read step_ion
            if (tid < cnt) {
                step_ion[4 * tid] = ions[3 * (w0 + tid)]; step_ion[4 * tid + 1] = ions[3 * (w0 + tid) + 1];
                step_ion[4 * tid + 2] = ions[3 * (w0 + tid) + 2]; step_ion[4 * tid + 3] = 1.f;
            }
            k_step(cnt);
        }
    } else {
        // candidates of every cell row, 32 at a time; non-members get weight 0 and contribute nothing
        for (int row = 0; row < ny_r * nz_r; ++row) {
            const int iy = rc.iy0 + row % ny_r, izc = rc.iz0 + row / ny_r;
            const int base = (izc * g.ny + iy) * g.nx;
            const uint32_t beg = p.cell_start[base + rc.ix0], end = p.cell_start[base + rc.ix1 + 1];
            for (uint32_t i0 = beg; i0 < end; i0 += kFspStep) {
                const int cnt = (int)min((uint32_t)kFspStep, end - i0);
                __syncthreads();
                if (tid < cnt) {
                    const float4 q = p.sorted[i0 + tid];
                    const float dx = __fsub_rn(q.x, cx), dy = __fsub_rn(q.y, cy), dz = __fsub_rn(q.z, cz);
                    step_ion[4 * tid] = dx; step_ion[4 * tid + 1] = dy; step_ion[4 * tid + 2] = dz;
                    step_ion[4 * tid + 3] = inside(dx, dy, dz, p.R2) ? 1.f : 0.f;
                }
                k_step(cnt);
            }
        }
    }
    // ---- |F| -> out[m][iz][iy][ix], four consecutive ix per thread ------------------------------------------------
    float *o = p.out + ((size_t)m * L + iz) * (size_t)L * L;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int iy = iy0 + 4 * ty + i;
        if (iy >= L) break;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int ix = ix0 + 4 * tx + j;
            if (ix < L) o[(size_t)iy * L + ix] = sqrtf(cr[i][j] * cr[i][j] + ci[i][j] * ci[i][j]);
        }
    }
  }
}

}  // namespace apx

using namespace apx;

extern "C" int apx_fsp_set_path(apx_plan *p, int32_t path)
{
    if (!p || (path != 0 && path != 1)) return APX_EINVAL;
    p->fsp_path = path;
    return APX_OK;
}

extern "C" int apx_fsp(apx_plan *p, const float *centres, int64_t M, float k_max, int32_t L, float *out, uint32_t *counts,
                       void *stream)
{
    if (!p || M < 0 || L < 1 || L > 1024 || !(k_max >= 0.0f) || !std::isfinite(k_max) || (M > 0 && (!centres || !out))) return APX_EINVAL;
    if (!p->ingested) return APX_ESTATE;
    if (M == 0) return APX_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != p->device) cudaSetDevice(p->device);
    auto done = [&](int code) { if (prev >= 0 && prev != p->device) cudaSetDevice(prev); return code; };
    auto cu = [&](cudaError_t e) { p->last_cuda = (int)e; return done(e == cudaErrorMemoryAllocation ? APX_ENOMEM : APX_ECUDA); };
    cudaStream_t st = (cudaStream_t)stream;
    // k axis (reading #25): L points over [-k_max, k_max], both ends included; fp64, rounded once
    if (L > p->cap_kaxis) {
        if (p->d_kaxis) cudaFree(p->d_kaxis);
        p->d_kaxis = nullptr; p->cap_kaxis = 0;
        cudaError_t e = cudaMalloc(&p->d_kaxis, sizeof(float) * L);
        if (e != cudaSuccess) return cu(e);
        p->cap_kaxis = L;
    }
    float kax[1024];
    for (int i = 0; i < L; ++i) kax[i] = L == 1 ? 0.0f : (float)(-(double)k_max + (double)i * (2.0 * (double)k_max / (double)(L - 1)));
    cudaError_t e = cudaMemcpyAsync(p->d_kaxis, kax, sizeof(float) * L, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cu(e);
    const int tiles = (L + kFspTile - 1) / kFspTile;
    const size_t smem = sizeof(float) * (4 * kFspStep * kFspTile + 4 * kFspStep + 3 * kFspCap);
    e = cudaFuncSetAttribute(k_fsp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cu(e);
    FspParams q;
    q.sorted = p->d_sorted; q.cell_start = p->d_cell_start; q.grid = p->d_grid; q.centres = centres; q.kaxis = p->d_kaxis;
    q.out = out; q.counts = counts; q.list = nullptr; q.L = L; q.tiles = tiles; q.R = p->R; q.R2 = p->R2;
    if (p->fsp_path == 1) {
        // FP32 pipe only
        const int64_t blocks = M * L * tiles * tiles;
        if (blocks > 0x7FFFFFFFLL) return done(APX_ERANGE);
        k_fsp<<<(unsigned)blocks, kFspThreads, smem, st>>>(q);
    } else {
        // tensor cores (fsp_mma.cu); the material points it leaves out (more ions than its shared buffer) are appended to a
        // device list and served by the FP32 kernel in the same stream
        if (M + 1 > p->cap_fsp_list) {
            if (p->d_fsp_list) cudaFree(p->d_fsp_list);
            p->d_fsp_list = nullptr; p->cap_fsp_list = 0;
            e = cudaMalloc(&p->d_fsp_list, (size_t)(M + 1) * 4);
            if (e != cudaSuccess) return cu(e);
            p->cap_fsp_list = M + 1;
        }
        e = cudaMemsetAsync(p->d_fsp_list, 0, 4, st);
        if (e != cudaSuccess) return cu(e);
        e = launch_fsp_mma(p, centres, M, L, L == 1 ? 0.0f : (float)(2.0 * (double)k_max / (double)(L - 1)), out, counts, p->d_fsp_list, st);
        if (e != cudaSuccess) return cu(e);
        q.list = p->d_fsp_list;
        k_fsp<<<(unsigned)(p->sm_count * 2), kFspThreads, smem, st>>>(q);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return cu(e);
    return done(APX_OK);
}

// ---- apx_fsp_noalloc: the same kernels with their scratch in a static device array (include/aptsig_ext.h) ------------------
//
// Layout of the array: [0, 4096) the k axis float32[<= 1024]; [4096, 4096 + 65792) the list uint32[1 + 16384] of the material
// points k_fsp_mma leaves to k_fsp (word 0 = count).  Every GPU that loads the library holds the array until exit.  In HOST
// code the name g_fsp_scratch is only a stand-in for the symbol, never a device address: the address each device uses is taken
// once per device with cudaGetSymbolAddress (below, with that device current) and handed to the kernels as an argument.
namespace apx {
constexpr int kNoAllocMaxM = APX_FSP_NOALLOC_MAX_M, kNoAllocMaxL = APX_FSP_NOALLOC_MAX_L;
constexpr size_t kNoAllocKaxisBytes = sizeof(float) * kNoAllocMaxL;                                     // 4096
constexpr size_t kNoAllocListBytes = ((sizeof(uint32_t) * (size_t)(1 + kNoAllocMaxM) + 255) / 256) * 256;      // 65792
static_assert(kNoAllocKaxisBytes % 256 == 0, "the list must start 256-byte aligned");
static_assert(kNoAllocKaxisBytes + kNoAllocListBytes == APX_FSP_NOALLOC_SCRATCH_BYTES, "header and layout disagree");
static __device__ __align__(256) unsigned char g_fsp_scratch[APX_FSP_NOALLOC_SCRATCH_BYTES];

// k axis (reading #25) exactly as apx_fsp computes it on the host -- fp64, every operation rounded on its own (no fused
// multiply-add), one final rounding to fp32 -- and the list count back to zero (the array keeps the previous call's contents).
__global__ void __launch_bounds__(1024) k_fsp_noalloc_prepare(unsigned char *scratch, float k_max, int L)
{
    float *kaxis = reinterpret_cast<float *>(scratch);
    uint32_t *list = reinterpret_cast<uint32_t *>(scratch + kNoAllocKaxisBytes);
    const int i = threadIdx.x;
    if (i < L) {
        const double step = L == 1 ? 0.0 : __ddiv_rn(__dmul_rn(2.0, (double)k_max), (double)(L - 1));
        kaxis[i] = L == 1 ? 0.0f : (float)__dadd_rn(-(double)k_max, __dmul_rn((double)i, step));
    }
    if (i == 0) list[0] = 0u;
}
}  // namespace apx

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_scratch_mu;
unsigned char *g_scratch_addr[kMaxDevices];      // device address of g_fsp_scratch on device d, nullptr = not resolved yet

// Device address of the scratch array on `device`, which must be the CURRENT device.  Resolved once per device.
cudaError_t scratch_address(int device, unsigned char **out)
{
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (!g_scratch_addr[device]) {
        void *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, apx::g_fsp_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch_addr[device] = static_cast<unsigned char *>(ptr);
    }
    *out = g_scratch_addr[device];
    return cudaSuccess;
}
}  // namespace

extern "C" int apx_fsp_noalloc_limits(int64_t *max_M, int32_t *max_L, int64_t *scratch_bytes)
{
    if (max_M) *max_M = kNoAllocMaxM;
    if (max_L) *max_L = kNoAllocMaxL;
    if (scratch_bytes) *scratch_bytes = APX_FSP_NOALLOC_SCRATCH_BYTES;
    return APX_OK;
}

extern "C" int apx_fsp_noalloc(apx_plan *p, const float *centres, int64_t M, float k_max, int32_t L, float *out, uint32_t *counts,
                               void *stream)
{
    if (!p || M < 0 || L < 1 || !(k_max >= 0.0f) || !std::isfinite(k_max) || (M > 0 && (!centres || !out))) return APX_EINVAL;
    if (M > kNoAllocMaxM || L > kNoAllocMaxL) return APX_ERANGE;          // beyond the static scratch: nothing is launched
    if (!p->ingested) return APX_ESTATE;
    if (M == 0) return APX_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != p->device) cudaSetDevice(p->device);
    auto done = [&](int code) { if (prev >= 0 && prev != p->device) cudaSetDevice(prev); return code; };
    auto cu = [&](cudaError_t e) { p->last_cuda = (int)e; return done(APX_ECUDA); };
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *scratch = nullptr;
    cudaError_t e = scratch_address(p->device, &scratch);                  // the plan's device is current here
    if (e != cudaSuccess) return cu(e);
    const float *kaxis = reinterpret_cast<const float *>(scratch);
    uint32_t *list = reinterpret_cast<uint32_t *>(scratch + kNoAllocKaxisBytes);
    const int tiles = (L + kFspTile - 1) / kFspTile;
    const size_t smem = sizeof(float) * (4 * kFspStep * kFspTile + 4 * kFspStep + 3 * kFspCap);
    e = cudaFuncSetAttribute(k_fsp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cu(e);
    const int64_t blocks = p->fsp_path == 1 ? M * L * tiles * tiles : M * ((L + 3) / 4) * tiles * tiles     /* k_fsp_mma: four z-slices per CTA */;
    if (blocks > 0x7FFFFFFFLL) return done(APX_ERANGE);
    k_fsp_noalloc_prepare<<<1, 1024, 0, st>>>(scratch, k_max, L);
    FspParams q;
    q.sorted = p->d_sorted; q.cell_start = p->d_cell_start; q.grid = p->d_grid; q.centres = centres; q.kaxis = kaxis;
    q.out = out; q.counts = counts; q.list = nullptr; q.L = L; q.tiles = tiles; q.R = p->R; q.R2 = p->R2;
    if (p->fsp_path == 1) {
        k_fsp<<<(unsigned)blocks, kFspThreads, smem, st>>>(q);
    } else {
        e = launch_fsp_mma_at(p, kaxis, centres, M, L, L == 1 ? 0.0f : (float)(2.0 * (double)k_max / (double)(L - 1)), out, counts,
                              list, st);
        if (e != cudaSuccess) return cu(e);
        q.list = list;
        k_fsp<<<(unsigned)(p->sm_count * 2), kFspThreads, smem, st>>>(q);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return cu(e);
    return done(APX_OK);
}
