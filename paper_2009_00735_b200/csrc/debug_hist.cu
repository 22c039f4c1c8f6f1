// debug_hist.cu -- test hook behind apx_debug_histograms: Eq. 1 histograms of one
// material point written to global memory, with the production gather (cell rows) and bin_of().
#include "common.cuh"

namespace apx {

__global__ void __launch_bounds__(256)
k_debug_hist(const float4 *__restrict__ sorted, const uint32_t *__restrict__ cell_start,
             const GridParams *__restrict__ gp, float cx, float cy, float cz,
             const float *__restrict__ dirs_scaled, int d0, uint32_t *__restrict__ out, int B, float R, float R2)
{
    const GridParams g = *gp;
    if (!g.n_accepted) return;
    const int d = d0 + blockIdx.x;
    uint32_t *hist = out + (size_t)blockIdx.x * B;
    const float npx = dirs_scaled[3 * d], npy = dirs_scaled[3 * d + 1], npz = dirs_scaled[3 * d + 2];
    const float half_b = (float)(B / 2), magic = magic_for(B);
    float mx = R * 1.00001f + fabsf(cx) * 1e-6f, my = R * 1.00001f + fabsf(cy) * 1e-6f, mz = R * 1.00001f + fabsf(cz) * 1e-6f;
    int ix0 = cell_coord(cx - mx, g.ox, g.inv_h, g.nx), ix1 = cell_coord(cx + mx, g.ox, g.inv_h, g.nx);
    int iy0 = cell_coord(cy - my, g.oy, g.inv_h, g.ny), iy1 = cell_coord(cy + my, g.oy, g.inv_h, g.ny);
    int iz0 = cell_coord(cz - mz, g.oz, g.inv_h, g.nz), iz1 = cell_coord(cz + mz, g.oz, g.inv_h, g.nz);
    for (int iz = iz0; iz <= iz1; ++iz)
        for (int iy = iy0; iy <= iy1; ++iy) {
            int base = (iz * g.ny + iy) * g.nx;
            uint32_t beg = cell_start[base + ix0], end = cell_start[base + ix1 + 1];
            for (uint32_t i = beg + threadIdx.x; i < end; i += blockDim.x) {
                float4 p = sorted[i];
                float dx = __fsub_rn(p.x, cx), dy = __fsub_rn(p.y, cy), dz = __fsub_rn(p.z, cz);
                if (inside(dx, dy, dz, R2)) atomicAdd(&hist[bin_of(npx, npy, npz, dx, dy, dz, half_b, magic)], 1u);
            }
        }
}

cudaError_t launch_debug_hist(Plan *p, const float *c, int d0, int nd, uint32_t *out, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(out, 0, (size_t)nd * p->B * sizeof(uint32_t), st);
    if (e != cudaSuccess || nd == 0) return e;
    k_debug_hist<<<nd, 256, 0, st>>>(p->d_sorted, p->d_cell_start, p->d_grid, c[0], c[1], c[2],
                                     p->d_dirs_scaled, d0, out, p->B, p->R, p->R2);
    return cudaGetLastError();
}

}  // namespace apx
