// refine.cu -- adaptive refinement of the ROI grid and the host-side
// orientation grid of the indexer (L367).
//   k_intensity_max : per material point max_d A_d / N_c (L210 "maximum intensity per signature", normalised, L424)
//   k_select        : ordered compaction of the material points with kappa_max >= kappa (L210: kappa >= 0.75)
//   k_centres       : split^3 new ROI centres per selected grid cell (L210: 5^3)
// Everything stays on the device; the selected count is read by k_centres from device memory, so the chain
// apx_query -> apx_intensity_max -> apx_refine_select -> apx_refine_centres enqueues without a host round trip.
#include <cmath>
#include <vector>
#include "common.cuh"
#include "../../include/aptsig_ext.h"

namespace apx {

// one warp per material point: coalesced float2 loads of the signature row, shuffle max
__global__ void __launch_bounds__(256)
k_intensity_max(const float2 *__restrict__ sig, const uint32_t *__restrict__ counts, int64_t M, int D, float *__restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const int64_t m = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (m >= M) return;
    const uint32_t n = counts[m];
    float best = 0.f;
    if (n) {
        const float2 *row = sig + m * D;
        for (int d = lane; d < D; d += 32) best = fmaxf(best, row[d].x);
#pragma unroll
        for (int o = 16; o; o >>= 1) best = fmaxf(best, __shfl_xor_sync(0xffffffffu, best, o));
        best = __fdiv_rn(best, (float)n);                       // max_d (A_d / N_c) = (max_d A_d) / N_c: division is monotone
    }
    if (lane == 0) out[m] = best;
}

// single CTA, ordered: tiles of 1024 material points, ballot + warp prefix + running base
__global__ void __launch_bounds__(1024)
k_select(const float *__restrict__ kappa_max, int64_t M, float kappa, uint32_t *__restrict__ selected, uint32_t *__restrict__ n_sel)
{
    __shared__ uint32_t warp_cnt[32];
    __shared__ uint32_t base;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) base = 0;
    __syncthreads();
    for (int64_t m0 = 0; m0 < M; m0 += 1024) {
        const int64_t m = m0 + threadIdx.x;
        const bool keep = m < M && kappa_max[m] >= kappa;
        const unsigned msk = __ballot_sync(0xffffffffu, keep);
        if (lane == 0) warp_cnt[wid] = __popc(msk);
        __syncthreads();
        uint32_t before = 0, total = 0;
        for (int w = 0; w < 32; ++w) {
            const uint32_t c = warp_cnt[w];
            if (w < wid) before += c;
            total += c;
        }
        if (keep) selected[base + before + __popc(msk & ((1u << lane) - 1u))] = (uint32_t)m;
        __syncthreads();
        if (threadIdx.x == 0) base += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_sel = base;
}

__global__ void __launch_bounds__(256)
k_centres(const float *__restrict__ centres, const uint32_t *__restrict__ selected, const uint32_t *__restrict__ n_sel,
          int64_t max_selected, int split, const float *__restrict__ offsets, float *__restrict__ out)
{
    const int64_t ns = min((int64_t)*n_sel, max_selected);
    const int s3 = split * split * split;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < ns * s3; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t s = t / s3;
        const int r = (int)(t % s3);
        const int ix = r % split, iy = (r / split) % split, iz = r / (split * split);
        const uint32_t m = selected[s];
        out[3 * t] = __fadd_rn(centres[3 * (size_t)m], offsets[ix]);
        out[3 * t + 1] = __fadd_rn(centres[3 * (size_t)m + 1], offsets[iy]);
        out[3 * t + 2] = __fadd_rn(centres[3 * (size_t)m + 2], offsets[iz]);
    }
}

}  // namespace apx

using namespace apx;

namespace {
struct Guard {
    int prev = -1;
    explicit Guard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); }
    ~Guard() { int cur = -1; if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev); }
};
int finish(apx_plan *p)
{
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) return APX_OK;
    p->last_cuda = (int)e;
    return APX_ECUDA;
}
}  // namespace

extern "C" int apx_intensity_max(apx_plan *p, const float *sig, const uint32_t *counts, int64_t M, float *kappa_max, void *stream)
{
    if (!p || M < 0 || (M > 0 && (!sig || !counts || !kappa_max))) return APX_EINVAL;
    if (M == 0) return APX_OK;
    Guard g(p->device);
    const int64_t threads = M * 32;
    k_intensity_max<<<(unsigned)((threads + 255) / 256), 256, 0, (cudaStream_t)stream>>>(reinterpret_cast<const float2 *>(sig), counts, M,
                                                                                        p->D, kappa_max);
    return finish(p);
}

extern "C" int apx_refine_select(apx_plan *p, const float *kappa_max, int64_t M, float kappa, uint32_t *selected,
                                 uint32_t *n_selected, void *stream)
{
    if (!p || M < 0 || !n_selected || (M > 0 && (!kappa_max || !selected))) return APX_EINVAL;
    if (M >= (1LL << 31)) return APX_ERANGE;
    Guard g(p->device);
    k_select<<<1, 1024, 0, (cudaStream_t)stream>>>(kappa_max, M, kappa, selected, n_selected);
    return finish(p);
}

extern "C" int apx_refine_centres(apx_plan *p, const float *centres, const uint32_t *selected, const uint32_t *n_selected,
                                  int64_t max_selected, float spacing, int32_t split, float *out, void *stream)
{
    if (!p || !n_selected || max_selected < 0 || split < 1 || split > 16 || !std::isfinite(spacing)) return APX_EINVAL;
    if (max_selected > 0 && (!centres || !selected || !out)) return APX_EINVAL;
    if (max_selected == 0) return APX_OK;
    Guard g(p->device);
    // sub-cell centre offsets: fp64, rounded once to fp32 (reading #21); passed through the plan's small scratch buffer
    float off[16];
    for (int i = 0; i < split; ++i) off[i] = (float)((((double)i + 0.5) / (double)split - 0.5) * (double)spacing);
    if (!p->d_refine_off) {
        cudaError_t e = cudaMalloc(&p->d_refine_off, sizeof(off));
        if (e != cudaSuccess) { p->last_cuda = (int)e; return APX_ENOMEM; }
    }
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(p->d_refine_off, off, sizeof(float) * split, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { p->last_cuda = (int)e; return APX_ECUDA; }
    k_centres<<<p->sm_count * 4, 256, 0, st>>>(centres, selected, n_selected, max_selected, split, p->d_refine_off, out);
    return finish(p);
}

// Orientation set (reading #23): Rodrigues lattice inside the m-3m fundamental zone, fp64 -> fp32 quaternions.
extern "C" int apx_so3_grid_cubic(float spacing_deg, float *quats, int64_t *Ng)
{
    if (!Ng || !(spacing_deg > 0.0f) || spacing_deg > 45.0f) return APX_EINVAL;
    const double h = std::tan((double)spacing_deg * M_PI / 180.0 / 2.0);
    const double lim = std::sqrt(2.0) - 1.0;
    const int n = (int)std::floor(lim / h + 1e-12);
    int64_t count = 0;
    for (int iz = -n; iz <= n; ++iz)
        for (int iy = -n; iy <= n; ++iy)
            for (int ix = -n; ix <= n; ++ix) {
                const double r[3] = {ix * h, iy * h, iz * h};
                const double amax = std::fmax(std::fabs(r[0]), std::fmax(std::fabs(r[1]), std::fabs(r[2])));
                if (amax > lim + 1e-12 || std::fabs(r[0]) + std::fabs(r[1]) + std::fabs(r[2]) > 1.0 + 1e-12) continue;
                if (quats) {
                    const double w = 1.0 / std::sqrt(1.0 + r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
                    quats[4 * count] = (float)w;
                    quats[4 * count + 1] = (float)(r[0] * w);
                    quats[4 * count + 2] = (float)(r[1] * w);
                    quats[4 * count + 3] = (float)(r[2] * w);
                }
                ++count;
            }
    *Ng = count;
    return APX_OK;
}
