// signature_fft.cu -- general signature kernel (any window, B = 256..4096): steps a2, a4-a7.
// One CTA = one material point x one chunk of directions.  The ROI's ions are gathered once into
// shared memory (SoA), then each warp takes one direction at a time: bins the ions into a private
// shared-memory histogram (Eq. 1), runs an in-place packed real FFT on it (the paper
// calls MKL/FFTW per histogram, L379; this is the hand-written batched replacement), scans the window
// for the largest |X_k|^2 (L75, L416) and stores (amplitude, bin).  Histograms never leave the SM.
#include "common.cuh"

namespace apx {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kDirChunk = 256;            // directions per CTA

// Gather (step a2): every warp walks x-rows of cells (contiguous in the sorted array), keeps ions with
// r^2 <= R2 and appends d = p - c to shared SoA arrays.  Returns the ROI ion count in *s_n (may exceed cap;
// then only the first cap are stored and the caller must use the streaming path).
__device__ __forceinline__ void gather_roi(const float4 *__restrict__ sorted, const uint32_t *__restrict__ cell_start,
                                           const GridParams &g, const RoiCells &rc, float cx, float cy, float cz,
                                           float R2, float *sx, float *sy, float *sz, int cap, int *s_n)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
    for (int row = wid; row < ny_r * nz_r; row += kWarps) {
        int iy = rc.iy0 + row % ny_r, iz = rc.iz0 + row / ny_r;
        int base = (iz * g.ny + iy) * g.nx;
        uint32_t beg = cell_start[base + rc.ix0], end = cell_start[base + rc.ix1 + 1];
        for (uint32_t i = beg + lane; i < ((end - beg + 31u) & ~31u) + beg; i += 32) {
            bool in = false;
            float dx = 0.f, dy = 0.f, dz = 0.f;
            if (i < end) {
                float4 p = sorted[i];
                dx = __fsub_rn(p.x, cx); dy = __fsub_rn(p.y, cy); dz = __fsub_rn(p.z, cz);
                in = inside(dx, dy, dz, R2);
            }
            unsigned m = __ballot_sync(0xffffffffu, in);
            if (m) {
                int pos = 0;
                if (lane == 0) pos = atomicAdd(s_n, __popc(m));
                pos = __shfl_sync(0xffffffffu, pos, 0) + __popc(m & ((1u << lane) - 1u));
                if (in && pos < cap) { sx[pos] = dx; sy[pos] = dy; sz[pos] = dz; }
            }
        }
    }
}

template <bool kStream>
__device__ __forceinline__ void bin_direction(uint32_t *hist, float npx, float npy, float npz, float half_b,
                                              float magic, const float *sx, const float *sy, const float *sz, int n,
                                              const float4 *__restrict__ sorted, const uint32_t *__restrict__ cell_start,
                                              const GridParams &g, const RoiCells &rc, float cx, float cy, float cz,
                                              float R2)
{
    const int lane = threadIdx.x & 31;
    if (!kStream) {
        for (int i = lane; i < n; i += 32)
            atomicAdd(&hist[bin_of(npx, npy, npz, sx[i], sy[i], sz[i], half_b, magic)], 1u);
    } else {
        // ROI larger than the shared-memory ion buffer: stream the cell rows again for every direction
        const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
        for (int row = 0; row < ny_r * nz_r; ++row) {
            int iy = rc.iy0 + row % ny_r, iz = rc.iz0 + row / ny_r;
            int base = (iz * g.ny + iy) * g.nx;
            uint32_t beg = cell_start[base + rc.ix0], end = cell_start[base + rc.ix1 + 1];
            for (uint32_t i = beg + lane; i < end; i += 32) {
                float4 p = sorted[i];
                float dx = __fsub_rn(p.x, cx), dy = __fsub_rn(p.y, cy), dz = __fsub_rn(p.z, cz);
                if (inside(dx, dy, dz, R2)) atomicAdd(&hist[bin_of(npx, npy, npz, dx, dy, dz, half_b, magic)], 1u);
            }
        }
    }
}

// In-place radix-2 decimation-in-frequency FFT of N = B/2 complex points held by one warp in shared
// memory; output in bit-reversed order.  tw[r] = exp(-2 pi i r / B), r < B/2.
__device__ __forceinline__ void warp_fft_dif(float2 *z, const float2 *__restrict__ tw, int N, int B)
{
    const int lane = threadIdx.x & 31;
    for (int half = N >> 1; half >= 1; half >>= 1) {
        const int tstep = B / (2 * half);
        for (int t = lane; t < (N >> 1); t += 32) {
            int pos = t & (half - 1);
            int i0 = ((t - pos) << 1) + pos;
            float2 a = z[i0], b = z[i0 + half];
            float2 w = tw[pos * tstep];
            float dr = a.x - b.x, di = a.y - b.y;
            z[i0] = make_float2(a.x + b.x, a.y + b.y);
            z[i0 + half] = make_float2(dr * w.x - di * w.y, dr * w.y + di * w.x);
        }
        __syncwarp();
    }
}

__global__ void __launch_bounds__(kThreads)
k_signature_fft(const float4 *__restrict__ sorted, const uint32_t *__restrict__ cell_start,
                const GridParams *__restrict__ gp, const float *__restrict__ centres,
                const float *__restrict__ dirs_scaled, const float2 *__restrict__ g_tw,
                float2 *__restrict__ sig, uint32_t *__restrict__ counts,
                int D, int B, int k_lo, int k_hi, float R, float R2, int cap, int nchunks,
                const uint32_t *__restrict__ list)
{
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t *s_hist = reinterpret_cast<uint32_t *>(smem);                       // [kWarps][B]
    float2 *s_tw = reinterpret_cast<float2 *>(s_hist + (size_t)kWarps * B);        // [B/2]
    float2 *s_res = s_tw + B / 2;                                                 // [kDirChunk]
    float *sx = reinterpret_cast<float *>(s_res + kDirChunk);                     // [cap] x3
    float *sy = sx + cap, *sz = sy + cap;
    __shared__ int s_n;

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < B / 2; i += kThreads) s_tw[i] = g_tw[i];
    // direct mode: one work item (material point, direction chunk) per CTA.  list mode: the grid is
    // persistent and walks the items of the material points named in list[1 .. list[0]].
    const int64_t n_items = list ? (int64_t)list[0] * nchunks : (int64_t)gridDim.x;
    for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int64_t m = list ? (int64_t)list[1 + item / nchunks] : item / nchunks;
    const int chunk = (int)(item % nchunks);
    const int d_begin = chunk * kDirChunk, d_end = min(D, d_begin + kDirChunk);
    const GridParams g = *gp;
    const float cx = centres[3 * m], cy = centres[3 * m + 1], cz = centres[3 * m + 2];
    const RoiCells rc = roi_cells(g, cx, cy, cz, R);

    __syncthreads();                 // previous item fully written out; s_tw loaded
    if (threadIdx.x == 0) s_n = 0;
    __syncthreads();
    if (g.n_accepted) gather_roi(sorted, cell_start, g, rc, cx, cy, cz, R2, sx, sy, sz, cap, &s_n);
    __syncthreads();
    const int n = s_n;
    if (chunk == 0 && threadIdx.x == 0 && counts) counts[m] = (uint32_t)n;
    const bool stream = n > cap;

    const int N = B >> 1;
    const int logN = 31 - __clz(N);
    const float half_b = (float)(B / 2), magic = magic_for(B);
    uint32_t *hist = s_hist + (size_t)wid * B;
    float *hf = reinterpret_cast<float *>(hist);
    float2 *z = reinterpret_cast<float2 *>(hist);

    for (int d = d_begin + wid; d < d_end; d += kWarps) {
        for (int j = lane; j < B; j += 32) hist[j] = 0u;
        __syncwarp();
        const float npx = dirs_scaled[3 * d], npy = dirs_scaled[3 * d + 1], npz = dirs_scaled[3 * d + 2];
        if (!stream)
            bin_direction<false>(hist, npx, npy, npz, half_b, magic, sx, sy, sz, n, sorted, cell_start, g, rc, cx, cy, cz, R2);
        else
            bin_direction<true>(hist, npx, npy, npz, half_b, magic, sx, sy, sz, n, sorted, cell_start, g, rc, cx, cy, cz, R2);
        __syncwarp();
        // counts -> float in place: z[j] = (h[2j], h[2j+1]) packs the real sequence into N complex points
        for (int j = lane; j < B; j += 32) hf[j] = (float)hist[j];
        __syncwarp();
        warp_fft_dif(z, s_tw, N, B);
        // unpack the window: X_k = (Z_k + conj Z_{N-k})/2 - i e^{-2 pi i k/B} (Z_k - conj Z_{N-k})/2
        float best = -1.0f;
        int kbest = k_lo;
        for (int k = k_lo + lane; k <= k_hi; k += 32) {
            int ka = k & (N - 1), kb = (N - k) & (N - 1);
            float2 za = z[__brev((unsigned)ka) >> (32 - logN)];
            float2 zb = z[__brev((unsigned)kb) >> (32 - logN)];
            float2 w = (k < N) ? s_tw[k] : make_float2(-1.0f, 0.0f);
            float er = za.x + zb.x, ei = za.y - zb.y;          // Z_k + conj Z_{N-k}
            float orr = za.x - zb.x, oi = za.y + zb.y;         // Z_k - conj Z_{N-k}
            // -i * w * (orr + i oi) = (w.y*orr + w.x*oi) + i (w.y*oi - w.x*orr)
            float xr = er + (w.y * orr + w.x * oi);
            float xi = ei + (w.y * oi - w.x * orr);
            float pw = xr * xr + xi * xi;                       // 4 |X_k|^2
            if (pw > best) { best = pw; kbest = k; }            // ascending k per lane: lowest k kept on ties
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            float ob = __shfl_xor_sync(0xffffffffu, best, o);
            int ok = __shfl_xor_sync(0xffffffffu, kbest, o);
            if (ob > best || (ob == best && ok < kbest)) { best = ob; kbest = ok; }
        }
        if (lane == 0) s_res[d - d_begin] = make_float2(0.5f * sqrtf(fmaxf(best, 0.0f)), (float)kbest);
        __syncwarp();
    }
    __syncthreads();
    float2 *out = sig + (size_t)m * D + d_begin;
    for (int i = threadIdx.x; i < d_end - d_begin; i += kThreads) out[i] = s_res[i];
    }
}

static int fft_cap_for(int B) { return B <= 1024 ? 3072 : (B == 2048 ? 2688 : 4096); }

static cudaError_t launch_fft_common(Plan *p, const float *centres, int64_t M, const uint32_t *list, float *sig,
                                     uint32_t *counts, cudaStream_t st)
{
    const int B = p->B, cap = fft_cap_for(B);
    const int nchunks = (p->D + kDirChunk - 1) / kDirChunk;
    size_t smem = (size_t)kWarps * B * 4 + (size_t)(B / 2) * 8 + (size_t)kDirChunk * 8 + (size_t)cap * 12;
    cudaError_t e = cudaFuncSetAttribute(k_signature_fft, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int64_t blocks = list ? (int64_t)p->sm_count * 2 : M * nchunks;
    if (blocks > 0x7FFFFFFFLL) return cudaErrorInvalidConfiguration;
    k_signature_fft<<<(unsigned)blocks, kThreads, smem, st>>>(
        p->d_sorted, p->d_cell_start, p->d_grid, centres, p->d_dirs_scaled, p->d_twiddle,
        reinterpret_cast<float2 *>(sig), counts, p->D, B, p->k_lo, p->k_hi, p->R, p->R2, cap, nchunks, list);
    return cudaGetLastError();
}

cudaError_t launch_signature_fft(Plan *p, const float *centres, int64_t M, float *sig, uint32_t *counts,
                                 cudaStream_t st)
{
    if (M == 0) return cudaSuccess;
    return launch_fft_common(p, centres, M, nullptr, sig, counts, st);
}

cudaError_t launch_signature_fft_list(Plan *p, const float *centres, const uint32_t *list, float *sig,
                                      uint32_t *counts, cudaStream_t st)
{
    return launch_fft_common(p, centres, 0, list, sig, counts, st);
}

}  // namespace apx
