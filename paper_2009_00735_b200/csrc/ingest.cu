// ingest.cu -- step a1: type filter + uniform cell-grid bucketing by a counting sort on the device.
// The paper queries ions with a tree (cost f R^3 rho log(V rho) per ROI);
// here a uniform grid with cell edge ~R/2 replaces it: ROIs are fixed-radius balls, so a grid gives
// contiguous x-rows of cells that are read with coalesced 16-byte loads.
// HBM-bound: 13 B read three times (bounds, count, scatter) + 16 B record written per ion = 55 B.
#include "common.cuh"

namespace apx {

// monotone float <-> int encoding for atomicMin/atomicMax on signed ints
__device__ __forceinline__ int f2ord(float f)
{
    int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7FFFFFFF;
}
__device__ __forceinline__ float ord2f(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7FFFFFFF); }

// Four consecutive ions (i4 a multiple of 4) per thread: three 16-byte loads for the coordinates and one 4-byte load for the
// types when the caller's arrays are aligned for it (vec), scalar loads otherwise and at the ragged end.  n = valid ions (0..4).
struct Ion4 {
    float x[4], y[4], z[4];
    uint32_t t[4];
    int n;
};
__device__ __forceinline__ Ion4 load_ion4(const float *__restrict__ xyz, const uint8_t *__restrict__ types, int64_t i4, int64_t N,
                                          bool vec_xyz, bool vec_types)
{
    Ion4 o;
    o.n = (int)min((int64_t)4, N - i4);
    if (o.n == 4 && vec_xyz) {
        const float4 a = *reinterpret_cast<const float4 *>(xyz + 3 * i4), b = *reinterpret_cast<const float4 *>(xyz + 3 * i4 + 4),
                     c = *reinterpret_cast<const float4 *>(xyz + 3 * i4 + 8);
        o.x[0] = a.x; o.y[0] = a.y; o.z[0] = a.z; o.x[1] = a.w; o.y[1] = b.x; o.z[1] = b.y;
        o.x[2] = b.z; o.y[2] = b.w; o.z[2] = c.x; o.x[3] = c.y; o.y[3] = c.z; o.z[3] = c.w;
    } else {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const bool ok = u < o.n;
            o.x[u] = ok ? xyz[3 * (i4 + u)] : 0.f; o.y[u] = ok ? xyz[3 * (i4 + u) + 1] : 0.f; o.z[u] = ok ? xyz[3 * (i4 + u) + 2] : 0.f;
        }
    }
    if (!types) {
#pragma unroll
        for (int u = 0; u < 4; ++u) o.t[u] = kUntyped;
    } else if (o.n == 4 && vec_types) {
        const uchar4 t = *reinterpret_cast<const uchar4 *>(types + i4);
        o.t[0] = t.x; o.t[1] = t.y; o.t[2] = t.z; o.t[3] = t.w;
    } else {
#pragma unroll
        for (int u = 0; u < 4; ++u) o.t[u] = u < o.n ? (uint32_t)types[i4 + u] : 0u;
    }
    return o;
}
// type filter + finite test on loaded values (has_types = the caller passed a type array)
__device__ __forceinline__ bool accepted_v(const uint32_t *mask, bool has_types, uint32_t t, float x, float y, float z)
{
    bool ok = true;
    if (has_types) ok = (mask[t >> 5] >> (t & 31)) & 1u;
    const float inf = __int_as_float(0x7f800000);
    return ok && fabsf(x) < inf && fabsf(y) < inf && fabsf(z) < inf;
}

__global__ void k_reset(GridParams *g)
{
    g->minx = g->miny = g->minz = 0x7FFFFFFF;
    g->maxx = g->maxy = g->maxz = (int)0x80000000;
    g->n_accepted = 0;
}

__global__ void __launch_bounds__(256) k_bounds(const float *__restrict__ xyz, const uint8_t *__restrict__ types,
                                                int64_t N, const uint32_t *__restrict__ mask, GridParams *g)
{
    int mn[3] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF};
    int mx[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
    unsigned cnt = 0;
    const bool vx = ((uintptr_t)xyz & 15) == 0, vt = ((uintptr_t)types & 3) == 0;
    for (int64_t i4 = 4 * (blockIdx.x * (int64_t)blockDim.x + threadIdx.x); i4 < N; i4 += 4 * (int64_t)gridDim.x * blockDim.x) {
        const Ion4 q = load_ion4(xyz, types, i4, N, vx, vt);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (u >= q.n || !accepted_v(mask, types != nullptr, q.t[u], q.x[u], q.y[u], q.z[u])) continue;
            ++cnt;
            const int ox = f2ord(q.x[u]), oy = f2ord(q.y[u]), oz = f2ord(q.z[u]);
            mn[0] = min(mn[0], ox); mn[1] = min(mn[1], oy); mn[2] = min(mn[2], oz);
            mx[0] = max(mx[0], ox); mx[1] = max(mx[1], oy); mx[2] = max(mx[2], oz);
        }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            mn[a] = min(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
            mx[a] = max(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
        }
        cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    }
    // block-level reduction in shared memory, then one set of global atomics per block
    __shared__ int s_mn[3], s_mx[3];
    __shared__ unsigned s_cnt;
    if (threadIdx.x == 0) {
        s_mn[0] = s_mn[1] = s_mn[2] = 0x7FFFFFFF;
        s_mx[0] = s_mx[1] = s_mx[2] = (int)0x80000000;
        s_cnt = 0;
    }
    __syncthreads();
    if ((threadIdx.x & 31) == 0 && cnt) {
#pragma unroll
        for (int a = 0; a < 3; ++a) { atomicMin(&s_mn[a], mn[a]); atomicMax(&s_mx[a], mx[a]); }
        atomicAdd(&s_cnt, cnt);
    }
    __syncthreads();
    if (threadIdx.x == 0 && s_cnt) {
        atomicMin(&g->minx, s_mn[0]); atomicMin(&g->miny, s_mn[1]); atomicMin(&g->minz, s_mn[2]);
        atomicMax(&g->maxx, s_mx[0]); atomicMax(&g->maxy, s_mx[1]); atomicMax(&g->maxz, s_mx[2]);
        atomicAdd(&g->n_accepted, s_cnt);
    }
}

// one thread: derive the grid from the bounds.  Cell edge h = R/2, doubled until the grid fits kMaxCells.
__global__ void k_grid_params(GridParams *g, float R)
{
    if (g->n_accepted == 0) {
        g->ox = g->oy = g->oz = 0.f; g->inv_h = 1.f; g->nx = g->ny = g->nz = 1; g->ncells = 1;
        return;
    }
    float lo[3] = {ord2f(g->minx), ord2f(g->miny), ord2f(g->minz)};
    float hi[3] = {ord2f(g->maxx), ord2f(g->maxy), ord2f(g->maxz)};
    float h = 0.5f * R;
    int n[3];
    for (;;) {
        double cells = 1.0;
        for (int a = 0; a < 3; ++a) {
            double e = ((double)hi[a] - (double)lo[a]) / (double)h;
            e = e < 2.0e9 ? e : 2.0e9;
            n[a] = (int)e + 1;
            cells *= (double)n[a];
        }
        if (cells <= (double)kMaxCells) break;
        h *= 2.0f;
    }
    g->ox = lo[0]; g->oy = lo[1]; g->oz = lo[2];
    g->inv_h = 1.0f / h;
    g->nx = n[0]; g->ny = n[1]; g->nz = n[2];
    g->ncells = n[0] * n[1] * n[2];
}

__global__ void __launch_bounds__(256) k_zero_cells(uint32_t *cell_start, const GridParams *g)
{
    int n = g->ncells + 1;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) cell_start[i] = 0;
}

// cell of an accepted ion, 0xFFFFFFFF for a rejected one (the same arithmetic in k_count and k_scatter: the scatter recomputes
// the cell instead of reading a cached id -- 8 B per ion less traffic and one dependent load less)
__device__ __forceinline__ uint32_t cell_of(const uint32_t *mask, bool has_types, uint32_t t, float x, float y, float z,
                                            float ox, float oy, float oz, float ih, int nx, int ny, int nz)
{
    if (!accepted_v(mask, has_types, t, x, y, z)) return 0xFFFFFFFFu;
    return (uint32_t)((cell_coord(z, oz, ih, nz) * ny + cell_coord(y, oy, ih, ny)) * nx + cell_coord(x, ox, ih, nx));
}

__global__ void __launch_bounds__(256) k_count(const float *__restrict__ xyz, const uint8_t *__restrict__ types,
                                               int64_t N, const uint32_t *__restrict__ mask,
                                               const GridParams *__restrict__ g, uint32_t *cell_count)
{
    const float ox = g->ox, oy = g->oy, oz = g->oz, ih = g->inv_h;
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const bool vx = ((uintptr_t)xyz & 15) == 0, vt = ((uintptr_t)types & 3) == 0;
    for (int64_t i4 = 4 * (blockIdx.x * (int64_t)blockDim.x + threadIdx.x); i4 < N; i4 += 4 * (int64_t)gridDim.x * blockDim.x) {
        const Ion4 q = load_ion4(xyz, types, i4, N, vx, vt);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (u >= q.n) continue;
            const uint32_t c = cell_of(mask, types != nullptr, q.t[u], q.x[u], q.y[u], q.z[u], ox, oy, oz, ih, nx, ny, nz);
            if (c != 0xFFFFFFFFu) atomicAdd(&cell_count[c], 1u);
        }
    }
}

// Exclusive scan of cell_count[0..ncells) in place, total at [ncells], in two fully parallel launches over tiles of 8192
// cells (8 consecutive cells per thread; the grid has at most 2^21 cells = 256 tiles):
//   k_scan_local: exclusive scan inside every tile, tile totals to tile_sum
//   k_scan_add  : every tile adds the sum of the totals of the tiles before it (<= 255 values, one block reduce)
constexpr int kScanItems = 8, kScanTile = 1024 * kScanItems;
__device__ __forceinline__ uint32_t block_exclusive(uint32_t tot, uint32_t *warp_sum, uint32_t *block_total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        uint32_t w = warp_sum[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += t;
        }
        warp_sum[lane] = wi - w;   // exclusive
        if (lane == 31) *block_total = wi;
    }
    __syncthreads();
    return warp_sum[wid] + inc - tot;
}
__global__ void __launch_bounds__(1024) k_scan_local(uint32_t *cell, uint32_t *tile_sum, const GridParams *g)
{
    __shared__ uint32_t warp_sum[32], total;
    const int n = g->ncells, i0 = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    if (blockIdx.x * kScanTile >= n) return;
    uint32_t v[kScanItems];
    const bool full = i0 + kScanItems <= n;                      // cell_start is 16-byte aligned and i0 a multiple of 8
    if (full) {
        const uint4 a = *reinterpret_cast<const uint4 *>(cell + i0), b4 = *reinterpret_cast<const uint4 *>(cell + i0 + 4);
        v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b4.x; v[5] = b4.y; v[6] = b4.z; v[7] = b4.w;
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) v[k] = i0 + k < n ? cell[i0 + k] : 0u;
    }
    uint32_t tot = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { const uint32_t t = v[k]; v[k] = tot; tot += t; }   // exclusive within the thread
    const uint32_t excl = block_exclusive(tot, warp_sum, &total);
    if (full) {
        *reinterpret_cast<uint4 *>(cell + i0) = make_uint4(excl + v[0], excl + v[1], excl + v[2], excl + v[3]);
        *reinterpret_cast<uint4 *>(cell + i0 + 4) = make_uint4(excl + v[4], excl + v[5], excl + v[6], excl + v[7]);
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k)
            if (i0 + k < n) cell[i0 + k] = excl + v[k];
    }
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}
__global__ void __launch_bounds__(1024) k_scan_add(uint32_t *cell, uint32_t *cursor, const uint32_t *tile_sum, const GridParams *g)
{
    __shared__ uint32_t warp_sum[32], before;
    const int n = g->ncells, tile = blockIdx.x, i0 = tile * kScanTile + threadIdx.x * kScanItems;
    if (tile * kScanTile >= n) return;
    block_exclusive((int)threadIdx.x < tile ? tile_sum[threadIdx.x] : 0u, warp_sum, &before);   // sum of the earlier tiles
    const uint32_t off = before;
    if (i0 + kScanItems <= n) {
        uint4 a = *reinterpret_cast<const uint4 *>(cell + i0), b4 = *reinterpret_cast<const uint4 *>(cell + i0 + 4);
        a.x += off; a.y += off; a.z += off; a.w += off; b4.x += off; b4.y += off; b4.z += off; b4.w += off;
        *reinterpret_cast<uint4 *>(cell + i0) = a; *reinterpret_cast<uint4 *>(cell + i0 + 4) = b4;
        *reinterpret_cast<uint4 *>(cursor + i0) = a; *reinterpret_cast<uint4 *>(cursor + i0 + 4) = b4;
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k)
            if (i0 + k < n) { const uint32_t val = cell[i0 + k] + off; cell[i0 + k] = val; cursor[i0 + k] = val; }
    }
    if (threadIdx.x == 0 && (tile + 1) * kScanTile >= n) cell[n] = off + tile_sum[tile];   // the last tile: grand total
}

// record = (x, y, z, ion type): the type lets one sorted copy serve several type masks (classes of a multi-signature plan)
__global__ void __launch_bounds__(256) k_scatter(const float *__restrict__ xyz, const uint8_t *__restrict__ types, int64_t N,
                                                 const uint32_t *__restrict__ mask, const GridParams *__restrict__ g,
                                                 uint32_t *cursor, float4 *__restrict__ sorted)
{
    const float ox = g->ox, oy = g->oy, oz = g->oz, ih = g->inv_h;
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const bool vx = ((uintptr_t)xyz & 15) == 0, vt = ((uintptr_t)types & 3) == 0;
    for (int64_t i4 = 4 * (blockIdx.x * (int64_t)blockDim.x + threadIdx.x); i4 < N; i4 += 4 * (int64_t)gridDim.x * blockDim.x) {
        const Ion4 q = load_ion4(xyz, types, i4, N, vx, vt);
        uint32_t c[4], pos[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            c[u] = u < q.n ? cell_of(mask, types != nullptr, q.t[u], q.x[u], q.y[u], q.z[u], ox, oy, oz, ih, nx, ny, nz) : 0xFFFFFFFFu;
#pragma unroll
        for (int u = 0; u < 4; ++u)                                  // four reservations in flight
            if (c[u] != 0xFFFFFFFFu) pos[u] = atomicAdd(&cursor[c[u]], 1u);
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (c[u] != 0xFFFFFFFFu) sorted[pos[u]] = make_float4(q.x[u], q.y[u], q.z[u], __uint_as_float(q.t[u]));
    }
}

cudaError_t launch_ingest(Plan *p, const float *xyz, const uint8_t *types, int64_t N, cudaStream_t st)
{
    const int blocks = p->sm_count * 8;
    k_reset<<<1, 1, 0, st>>>(p->d_grid);
    if (N > 0) k_bounds<<<blocks, 256, 0, st>>>(xyz, types, N, p->d_type_mask, p->d_grid);
    k_grid_params<<<1, 1, 0, st>>>(p->d_grid, p->R);
    k_zero_cells<<<blocks, 256, 0, st>>>(p->d_cell_start, p->d_grid);
    if (N > 0)
        k_count<<<blocks, 256, 0, st>>>(xyz, types, N, p->d_type_mask, p->d_grid, p->d_cell_start);
    k_scan_local<<<kMaxCells / kScanTile, 1024, 0, st>>>(p->d_cell_start, p->d_scan_tiles, p->d_grid);
    k_scan_add<<<kMaxCells / kScanTile, 1024, 0, st>>>(p->d_cell_start, p->d_cell_cursor, p->d_scan_tiles, p->d_grid);
    if (N > 0) k_scatter<<<blocks, 256, 0, st>>>(xyz, types, N, p->d_type_mask, p->d_grid, p->d_cell_cursor, p->d_sorted);
    return cudaGetLastError();
}

}  // namespace apx
