// index.cu -- indexing of signatures against rotated references (Eq. 3).
//
// Pre-processing, once per (candidate, orientation set), apx_indexer_create:
//   * the n_hat strongest nodes of the normalised reference image (L369 "pick those nodes for which the signal is
//     strongest", decreasing order, lower node index first among equals) -- host, a sort of D numbers;
//   * the look-up table p[g][v] = mesh node closest to node v rotated by orientation g (L369-371), built on the device by
//     k_lut_build: fp64 rotation of the node by the unit quaternion (v' = q v q*), nearest node = largest fp64 dot product,
//     lowest index on ties.  Candidates come from a uniform 3-D cell grid over [-1,1]^3 (cell edge e): a node within
//     chord distance e of the query lies in the 3x3x3 cells around it, so if the best candidate is that close it is the
//     true nearest node; otherwise the thread falls back to all D nodes (never on the grids of the paper).
// Indexing, apx_index (L371-373, L395: N_roi x N_g x n_hat gathers):
//   * k_img_transpose: normalised intensities A / N_c (reading #19) of a chunk of material points, transposed so that the
//     32 material points of a block are the 32 lanes of a warp: imgT[block][node][lane].  One gather of the table then
//     reads ONE 128-byte line for 32 (material point, orientation, node) triples -- L2-bound, fully coalesced.
//   * k_index: CTA = 8 warps = 8 blocks of 32 material points x a range of orientations; the table rows of a batch of
//     orientations are staged in shared memory once per CTA and read as warp-uniform LDS.128 (8 node indices each);
//     Delta = sum_v (S_msr[p_v^g] - S_ref[v])^2 accumulated in fp32 per lane; every lane keeps its K best (Delta, g).
//   * k_index_merge: the per-range lists of a material point are merged into the K best overall (smallest Delta, lowest
//     orientation index among equals).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>
#include <vector>
#include <cuda_runtime.h>
#include "../../include/aptsig_ext.h"

namespace {

constexpr int kMaxK = APX_INDEX_MAX_K;
constexpr int kIdxWarps = 8;                    // material-point blocks per CTA
constexpr int kGBatch = 4;                      // table rows staged per batch
constexpr int64_t kChunkPoints = 2048;          // material points transposed and indexed per pass

struct Indexer {
    int device, D, n_hat, n_hat_pad, sm_count;
    int64_t Ng;
    int last_cuda;
    float *d_dirs;          // [D][3]
    float *d_quats;         // [Ng][4]
    int *d_nodes;           // [n_hat]
    float *d_ref;           // [n_hat_pad] reference intensity of the strongest nodes (padding 0)
    uint32_t *d_lut;        // [Ng][n_hat_pad] (padding repeats node 0 of the row with reference = its own value: see k_index)
    int *d_cell_start;      // [nc^3 + 1]
    int *d_cell_nodes;      // [D]
    int nc;                 // cells per axis
    float *d_imgT;          // [chunk/32][D][32]
    int64_t cap_img_points;
    float *d_part_delta;    // [chunk][ranges][kMaxK]
    int *d_part_g;
    int64_t cap_part;
    std::vector<int> h_nodes;
    std::vector<float> h_ref;
};

// ---- look-up table ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int cell_of(double v, int nc)
{
    int c = (int)floor((v + 1.0) * 0.5 * nc);
    return min(max(c, 0), nc - 1);
}

__global__ void __launch_bounds__(256)
k_lut_build(const float *__restrict__ dirs, int D, const float *__restrict__ quats, int64_t Ng, const int *__restrict__ nodes,
            int n_hat, int n_hat_pad, const int *__restrict__ cell_start, const int *__restrict__ cell_nodes, int nc,
            uint32_t *__restrict__ lut)
{
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= Ng * n_hat_pad) return;
    const int64_t g = t / n_hat_pad;
    const int v = (int)(t % n_hat_pad);
    if (v >= n_hat) { lut[t] = 0xFFFFFFFFu; return; }      // padding entry: skipped by k_index
    const double w = quats[4 * g], x = quats[4 * g + 1], y = quats[4 * g + 2], z = quats[4 * g + 3];
    const int node = nodes[v];
    const double nx = dirs[3 * node], ny = dirs[3 * node + 1], nz = dirs[3 * node + 2];
    // active rotation v' = q v q* written as the rotation matrix of (w, x, y, z)
    const double rx = (1 - 2 * (y * y + z * z)) * nx + 2 * (x * y - z * w) * ny + 2 * (x * z + y * w) * nz;
    const double ry = 2 * (x * y + z * w) * nx + (1 - 2 * (x * x + z * z)) * ny + 2 * (y * z - x * w) * nz;
    const double rz = 2 * (x * z - y * w) * nx + 2 * (y * z + x * w) * ny + (1 - 2 * (x * x + y * y)) * nz;
    double best = -4.0;
    int jbest = 0;
    auto consider = [&](int j) {
        const double d = (double)dirs[3 * j] * rx + (double)dirs[3 * j + 1] * ry + (double)dirs[3 * j + 2] * rz;
        if (d > best || (d == best && j < jbest)) { best = d; jbest = j; }
    };
    const int cx = cell_of(rx, nc), cy = cell_of(ry, nc), cz = cell_of(rz, nc);
    for (int iz = max(cz - 1, 0); iz <= min(cz + 1, nc - 1); ++iz)
        for (int iy = max(cy - 1, 0); iy <= min(cy + 1, nc - 1); ++iy)
            for (int ix = max(cx - 1, 0); ix <= min(cx + 1, nc - 1); ++ix) {
                const int c = (iz * nc + iy) * nc + ix;
                for (int i = cell_start[c]; i < cell_start[c + 1]; ++i) consider(cell_nodes[i]);
            }
    // chord^2 = |n|^2 + |r|^2 - 2 n.r <= e^2 guarantees that no node outside the 27 cells is closer (margin for |n| != 1)
    const double e = 2.0 / nc;
    if (!(2.0 - 2.0 * best <= 0.9 * e * e)) {
        best = -4.0; jbest = 0;
        for (int j = 0; j < D; ++j) consider(j);
    }
    lut[t] = (uint32_t)jbest;
}

// ---- normalise + transpose a chunk of measured signatures ---------------------------------------------------------
// sig [M][D][2] (amplitude at [..][0]) -> imgT[(m - m0) / 32][d][(m - m0) % 32] = A / N_c (0 for an empty ROI, or A itself
// when counts == nullptr: the caller has normalised).  Tile transpose through shared memory: coalesced on both sides.
__global__ void __launch_bounds__(256)
k_img_transpose(const float2 *__restrict__ sig, const uint32_t *__restrict__ counts, int64_t m0, int64_t M, int D,
                float *__restrict__ imgT)
{
    __shared__ float tile[32][33];
    const int64_t blk = blockIdx.y;                               // block of 32 material points within the chunk
    const int d0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;       // 32 x 8
    for (int r = ty; r < 32; r += 8) {                            // row r = material point, column tx = node
        const int64_t m = m0 + blk * 32 + r;
        float v = 0.f;
        if (m < M && d0 + tx < D) {
            const float a = sig[m * D + d0 + tx].x;
            if (counts) {
                const uint32_t n = counts[m];
                v = n ? __fdiv_rn(a, (float)n) : 0.f;
            } else {
                v = a;
            }
        }
        tile[r][tx] = v;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8)                              // row r = node, column tx = material point (lane)
        if (d0 + r < D) imgT[(blk * D + d0 + r) * 32 + tx] = tile[tx][r];
}

// ---- Eq. 3 ----------------------------------------------------------------------------------------------------------
struct TopK {
    float d[kMaxK];
    int g[kMaxK];
};
__device__ __forceinline__ void topk_insert(TopK &t, int K, float delta, int g)
{
    // sorted ascending by (delta, g); orientations arrive in increasing g, so a tie never displaces an earlier entry
    if (!(delta < t.d[K - 1])) return;
    int i = K - 1;
#pragma unroll
    for (int s = kMaxK - 1; s > 0; --s) {
        if (s <= i && t.d[s - 1] > delta) { t.d[s] = t.d[s - 1]; t.g[s] = t.g[s - 1]; i = s - 1; }
    }
    t.d[i] = delta; t.g[i] = g;
}

__global__ void __launch_bounds__(kIdxWarps * 32)
k_index(const float *__restrict__ imgT, const uint32_t *__restrict__ lut, const float *__restrict__ ref, int D, int n_hat_pad,
        int64_t Ng, int nranges, int64_t n_blocks, int K, float *__restrict__ part_delta, int *__restrict__ part_g)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *s_ref = reinterpret_cast<float *>(smem_raw);                              // [n_hat_pad]
    uint32_t *s_lut = reinterpret_cast<uint32_t *>(s_ref + n_hat_pad);                // [2][kGBatch][n_hat_pad]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int range = blockIdx.x;                                                    // orientation range (fastest: CTAs that
    const int64_t blk = (int64_t)blockIdx.y * kIdxWarps + warp;                       //  run together share the image blocks)
    const int64_t g_begin = Ng * range / nranges, g_end = Ng * (range + 1) / nranges;
    for (int i = tid; i < n_hat_pad; i += blockDim.x) s_ref[i] = ref[i];
    const bool active = blk < n_blocks;
    const float *img = imgT + (active ? blk : 0) * (int64_t)D * 32 + lane;
    TopK best;
#pragma unroll
    for (int s = 0; s < kMaxK; ++s) { best.d[s] = __int_as_float(0x7f800000); best.g[s] = -1; }

    auto stage = [&](int buf, int64_t g0) {                                          // rows [g0, g0 + kGBatch) -> s_lut[buf]
        const int64_t n = min((int64_t)kGBatch, g_end - g0) * n_hat_pad;
        const uint4 *src = reinterpret_cast<const uint4 *>(lut + g0 * n_hat_pad);
        uint4 *dst = reinterpret_cast<uint4 *>(s_lut + (size_t)buf * kGBatch * n_hat_pad);
        for (int64_t i = tid; i < n / 4; i += blockDim.x) dst[i] = src[i];
    };
    if (g_begin < g_end) stage(0, g_begin);
    __syncthreads();
    int buf = 0;
    for (int64_t g0 = g_begin; g0 < g_end; g0 += kGBatch, buf ^= 1) {
        if (g0 + kGBatch < g_end) stage(buf ^ 1, g0 + kGBatch);                      // next batch while this one is used
        const int nb = (int)min((int64_t)kGBatch, g_end - g0);
        if (active) {
            for (int j = 0; j < nb; ++j) {
                const uint4 *row = reinterpret_cast<const uint4 *>(s_lut + ((size_t)buf * kGBatch + j) * n_hat_pad);
                const float4 *rf = reinterpret_cast<const float4 *>(s_ref);
                float acc0 = 0.f, acc1 = 0.f;
                for (int v4 = 0; v4 < n_hat_pad / 4; v4 += 2) {                       // 8 nodes per iteration
                    const uint4 ia = row[v4], ib = row[v4 + 1];
                    const float4 ra = rf[v4], rb = rf[v4 + 1];
                    // padding entries (0xFFFFFFFF) contribute nothing
                    const float a0 = ia.x != 0xFFFFFFFFu ? __ldg(img + (size_t)ia.x * 32) - ra.x : 0.f;
                    const float a1 = ia.y != 0xFFFFFFFFu ? __ldg(img + (size_t)ia.y * 32) - ra.y : 0.f;
                    const float a2 = ia.z != 0xFFFFFFFFu ? __ldg(img + (size_t)ia.z * 32) - ra.z : 0.f;
                    const float a3 = ia.w != 0xFFFFFFFFu ? __ldg(img + (size_t)ia.w * 32) - ra.w : 0.f;
                    const float b0 = ib.x != 0xFFFFFFFFu ? __ldg(img + (size_t)ib.x * 32) - rb.x : 0.f;
                    const float b1 = ib.y != 0xFFFFFFFFu ? __ldg(img + (size_t)ib.y * 32) - rb.y : 0.f;
                    const float b2 = ib.z != 0xFFFFFFFFu ? __ldg(img + (size_t)ib.z * 32) - rb.z : 0.f;
                    const float b3 = ib.w != 0xFFFFFFFFu ? __ldg(img + (size_t)ib.w * 32) - rb.w : 0.f;
                    acc0 = fmaf(a0, a0, acc0); acc1 = fmaf(a1, a1, acc1); acc0 = fmaf(a2, a2, acc0); acc1 = fmaf(a3, a3, acc1);
                    acc0 = fmaf(b0, b0, acc0); acc1 = fmaf(b1, b1, acc1); acc0 = fmaf(b2, b2, acc0); acc1 = fmaf(b3, b3, acc1);
                }
                topk_insert(best, K, acc0 + acc1, (int)(g0 + j));
            }
        }
        __syncthreads();                                                             // next batch staged, this one consumed
    }
    if (active) {
        const int64_t m = blk * 32 + lane;                                           // material point within the chunk
        for (int s = 0; s < K; ++s) {
            part_delta[(m * nranges + range) * kMaxK + s] = best.d[s];
            part_g[(m * nranges + range) * kMaxK + s] = best.g[s];
        }
    }
}

// one thread per material point: merge the per-range lists (each sorted; ranges ordered by orientation index)
__global__ void __launch_bounds__(128)
k_index_merge(const float *__restrict__ part_delta, const int *__restrict__ part_g, int64_t n_points, int nranges, int K,
              float *__restrict__ best_delta, int *__restrict__ best_g)
{
    const int64_t m = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (m >= n_points) return;
    TopK best;
#pragma unroll
    for (int s = 0; s < kMaxK; ++s) { best.d[s] = __int_as_float(0x7f800000); best.g[s] = -1; }
    for (int r = 0; r < nranges; ++r)
        for (int s = 0; s < K; ++s) {
            const int g = part_g[(m * nranges + r) * kMaxK + s];
            if (g >= 0) topk_insert(best, K, part_delta[(m * nranges + r) * kMaxK + s], g);
        }
    for (int s = 0; s < K; ++s) { best_delta[m * K + s] = best.d[s]; best_g[m * K + s] = best.g[s]; }
}

#define CUI(ix, call)                                 \
    do {                                              \
        cudaError_t e__ = (call);                     \
        if (e__ != cudaSuccess) {                     \
            (ix)->last_cuda = (int)e__;               \
            return e__ == cudaErrorMemoryAllocation ? APX_ENOMEM : APX_ECUDA; \
        }                                             \
    } while (0)

struct DevGuard {
    int prev = -1;
    explicit DevGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); }
    ~DevGuard() { int cur = -1; if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev); }
};

}  // namespace

struct apx_indexer : public Indexer {};

extern "C" int apx_indexer_destroy(apx_indexer *ix)
{
    if (!ix) return APX_OK;
    DevGuard guard(ix->device);
    void *bufs[] = {ix->d_dirs, ix->d_quats, ix->d_nodes, ix->d_ref, ix->d_lut, ix->d_cell_start, ix->d_cell_nodes, ix->d_imgT,
                    ix->d_part_delta, ix->d_part_g};
    for (void *b : bufs)
        if (b) cudaFree(b);
    delete ix;
    return APX_OK;
}

extern "C" int apx_indexer_create(const float *dirs, int32_t D, const float *quats, int64_t Ng, const float *ref_image,
                                  int32_t n_hat, int32_t device, apx_indexer **out)
{
    if (!out) return APX_EINVAL;
    *out = nullptr;
    if (!dirs || !quats || !ref_image || D < 1 || Ng < 1 || n_hat < 1 || n_hat > D) return APX_EINVAL;
    if (Ng >= (1LL << 31)) return APX_ERANGE;
    apx_indexer *ix = new (std::nothrow) apx_indexer();
    if (!ix) return APX_ENOMEM;
    ix->device = device; ix->D = D; ix->Ng = Ng; ix->n_hat = n_hat; ix->n_hat_pad = (n_hat + 7) & ~7; ix->last_cuda = 0;
    ix->d_dirs = ix->d_quats = ix->d_ref = ix->d_imgT = ix->d_part_delta = nullptr;
    ix->d_nodes = ix->d_cell_start = ix->d_cell_nodes = ix->d_part_g = nullptr;
    ix->d_lut = nullptr; ix->cap_img_points = 0; ix->cap_part = 0;
    DevGuard guard(device);
    auto fail = [&](int code) { apx_indexer_destroy(ix); return code; };
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return fail(APX_ECUDA);
    ix->sm_count = prop.multiProcessorCount;

    // strongest nodes of the reference, decreasing, lower index first among equals (L369)
    std::vector<int> order(D);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return ref_image[a] > ref_image[b]; });
    ix->h_nodes.assign(order.begin(), order.begin() + n_hat);
    ix->h_ref.assign(ix->n_hat_pad, 0.f);
    for (int v = 0; v < n_hat; ++v) ix->h_ref[v] = ref_image[ix->h_nodes[v]];

    // 3-D cell grid over [-1,1]^3 for the nearest-node search: cell edge ~ 2.5 mean node spacings
    const double spacing = std::sqrt(4.0 * M_PI / (double)D);
    int nc = (int)std::floor(2.0 / (2.5 * spacing));
    nc = std::max(1, std::min(nc, 128));
    ix->nc = nc;
    std::vector<int> cell_of_node(D), cell_start((size_t)nc * nc * nc + 1, 0), cell_nodes(D);
    auto cell1 = [&](double v) { int c = (int)std::floor((v + 1.0) * 0.5 * nc); return std::min(std::max(c, 0), nc - 1); };
    for (int j = 0; j < D; ++j) {
        cell_of_node[j] = (cell1(dirs[3 * j + 2]) * nc + cell1(dirs[3 * j + 1])) * nc + cell1(dirs[3 * j]);
        ++cell_start[cell_of_node[j] + 1];
    }
    for (size_t c = 0; c + 1 < cell_start.size(); ++c) cell_start[c + 1] += cell_start[c];
    {
        std::vector<int> cur(cell_start.begin(), cell_start.end() - 1);
        for (int j = 0; j < D; ++j) cell_nodes[cur[cell_of_node[j]]++] = j;         // ascending node index inside a cell
    }
#define CUF(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { ix->last_cuda = (int)e__; \
        return fail(e__ == cudaErrorMemoryAllocation ? APX_ENOMEM : APX_ECUDA); } } while (0)
    CUF(cudaMalloc(&ix->d_dirs, (size_t)D * 12));
    CUF(cudaMalloc(&ix->d_quats, (size_t)Ng * 16));
    CUF(cudaMalloc(&ix->d_nodes, (size_t)n_hat * 4));
    CUF(cudaMalloc(&ix->d_ref, (size_t)ix->n_hat_pad * 4));
    CUF(cudaMalloc(&ix->d_lut, (size_t)Ng * ix->n_hat_pad * 4));
    CUF(cudaMalloc(&ix->d_cell_start, cell_start.size() * 4));
    CUF(cudaMalloc(&ix->d_cell_nodes, (size_t)D * 4));
    CUF(cudaMemcpy(ix->d_dirs, dirs, (size_t)D * 12, cudaMemcpyHostToDevice));
    CUF(cudaMemcpy(ix->d_quats, quats, (size_t)Ng * 16, cudaMemcpyHostToDevice));
    CUF(cudaMemcpy(ix->d_nodes, ix->h_nodes.data(), (size_t)n_hat * 4, cudaMemcpyHostToDevice));
    CUF(cudaMemcpy(ix->d_ref, ix->h_ref.data(), (size_t)ix->n_hat_pad * 4, cudaMemcpyHostToDevice));
    CUF(cudaMemcpy(ix->d_cell_start, cell_start.data(), cell_start.size() * 4, cudaMemcpyHostToDevice));
    CUF(cudaMemcpy(ix->d_cell_nodes, cell_nodes.data(), (size_t)D * 4, cudaMemcpyHostToDevice));
    const int64_t total = Ng * ix->n_hat_pad;
    k_lut_build<<<(unsigned)((total + 255) / 256), 256>>>(ix->d_dirs, D, ix->d_quats, Ng, ix->d_nodes, n_hat, ix->n_hat_pad,
                                                         ix->d_cell_start, ix->d_cell_nodes, nc, ix->d_lut);
    CUF(cudaGetLastError());
    CUF(cudaDeviceSynchronize());
#undef CUF
    *out = ix;
    return APX_OK;
}

extern "C" int apx_indexer_nodes(const apx_indexer *ix, int32_t *nodes, float *ref_values)
{
    if (!ix) return APX_EINVAL;
    if (nodes) std::memcpy(nodes, ix->h_nodes.data(), (size_t)ix->n_hat * 4);
    if (ref_values) std::memcpy(ref_values, ix->h_ref.data(), (size_t)ix->n_hat * 4);
    return APX_OK;
}

extern "C" int apx_indexer_lut(apx_indexer *ix, int64_t g0, int64_t ng, int32_t *out)
{
    if (!ix || g0 < 0 || ng < 0 || g0 + ng > ix->Ng || (ng > 0 && !out)) return APX_EINVAL;
    DevGuard guard(ix->device);
    // rows are padded to a multiple of 8 entries on the device; copy the n_hat real entries of every row
    CUI(ix, cudaMemcpy2D(out, (size_t)ix->n_hat * 4, ix->d_lut + g0 * ix->n_hat_pad, (size_t)ix->n_hat_pad * 4,
                         (size_t)ix->n_hat * 4, (size_t)ng, cudaMemcpyDeviceToHost));
    return APX_OK;
}

extern "C" int apx_last_cuda_error_indexer(const apx_indexer *ix) { return ix ? ix->last_cuda : (int)cudaErrorInvalidValue; }

extern "C" int apx_index(apx_indexer *ix, const float *sig, const uint32_t *counts, int64_t M, int32_t K, float *best_delta,
                         int32_t *best_g, void *stream)
{
    if (!ix || M < 0 || K < 1 || K > kMaxK || (int64_t)K > ix->Ng || (M > 0 && (!sig || !best_delta || !best_g))) return APX_EINVAL;
    if (M == 0) return APX_OK;
    DevGuard guard(ix->device);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t chunk = std::min<int64_t>(M, kChunkPoints);
    // orientation ranges: as many CTAs along the fastest grid axis as the machine holds at a time (six per SM: shared memory),
    // so that the resident CTAs all work on ONE row of 8 image blocks (8 x D x 128 B = 42 MB at D = 40 962) and the gathers hit
    // in L2; with two ranges per SM three rows (126 MB) were resident at once and 39 % of the sectors came from DRAM
    int per_sm = 6;
    if (const char *ev = std::getenv("APX_TUNE_INDEX_RANGES")) per_sm = std::max(1, std::atoi(ev));
    int nranges = (int)std::min<int64_t>(ix->Ng, (int64_t)ix->sm_count * per_sm);
    if (chunk > ix->cap_img_points) {
        if (ix->d_imgT) cudaFree(ix->d_imgT);
        ix->d_imgT = nullptr; ix->cap_img_points = 0;
        CUI(ix, cudaMalloc(&ix->d_imgT, (size_t)((chunk + 31) / 32) * ix->D * 32 * 4));
        ix->cap_img_points = chunk;
    }
    const int64_t need_part = ((chunk + 31) / 32) * 32 * nranges * kMaxK;
    if (need_part > ix->cap_part) {
        if (ix->d_part_delta) cudaFree(ix->d_part_delta);
        if (ix->d_part_g) cudaFree(ix->d_part_g);
        ix->d_part_delta = nullptr; ix->d_part_g = nullptr; ix->cap_part = 0;
        CUI(ix, cudaMalloc(&ix->d_part_delta, (size_t)need_part * 4));
        CUI(ix, cudaMalloc(&ix->d_part_g, (size_t)need_part * 4));
        ix->cap_part = need_part;
    }
    const size_t smem = (size_t)ix->n_hat_pad * 4 + (size_t)2 * kGBatch * ix->n_hat_pad * 4;
    CUI(ix, cudaFuncSetAttribute(k_index, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    for (int64_t m0 = 0; m0 < M; m0 += chunk) {
        const int64_t mc = std::min(chunk, M - m0);
        const int64_t n_blocks = (mc + 31) / 32;
        dim3 tg((unsigned)((ix->D + 31) / 32), (unsigned)n_blocks);
        k_img_transpose<<<tg, 256, 0, st>>>(reinterpret_cast<const float2 *>(sig), counts, m0, M, ix->D, ix->d_imgT);
        dim3 grid((unsigned)nranges, (unsigned)((n_blocks + kIdxWarps - 1) / kIdxWarps));
        k_index<<<grid, kIdxWarps * 32, smem, st>>>(ix->d_imgT, ix->d_lut, ix->d_ref, ix->D, ix->n_hat_pad, ix->Ng, nranges,
                                                   n_blocks, K, ix->d_part_delta, ix->d_part_g);
        k_index_merge<<<(unsigned)((mc + 127) / 128), 128, 0, st>>>(ix->d_part_delta, ix->d_part_g, mc, nranges, K,
                                                                   best_delta + m0 * K, best_g + m0 * K);
        CUI(ix, cudaGetLastError());
    }
    return APX_OK;
}
