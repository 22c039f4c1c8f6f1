// common.cuh -- internal declarations shared by the libaptsig translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/aptsig.h"

namespace apx {

// Uniform cell grid over the accepted ions; lives in DEVICE memory and is written by k_grid_params,
// so that ingest never synchronises with the host.
struct GridParams {
    float ox, oy, oz;      // origin = min corner of the accepted ions
    float inv_h;           // 1 / cell edge
    int nx, ny, nz;        // cells per axis (x fastest in the cell index)
    int ncells;            // nx*ny*nz  (<= kMaxCells)
    unsigned n_accepted;   // ions that passed the type / finite filter
    // ordered-int encodings of min/max used by the bounds reduction
    int minx, miny, minz, maxx, maxy, maxz;
};

constexpr int kMaxCells = 1 << 21;

// Signatures of one plan ("multiple signatures (for different atom types) are computed per
// ROI", L126-130, L208 "several lattice plane families {002}, {220}, {111}", L416-418): up to kMaxSpecs (type mask, spectral
// window, peak mode, normalisation) tuples served by ONE ingest and one launch.  Specs with the same type mask form a class:
// a class is gathered and binned once, its histograms transformed once over the union window [plan k_lo, plan k_hi], and
// every spec of the class picks its peak from its own sub-window.
constexpr int kMaxSpecs = APX_MAX_SIGNATURES;
constexpr uint32_t kUntyped = 0xFFFFu;      // type stored for ions ingested without a type array: accepted by every class
struct SpecSet {
    int n_specs, n_classes;
    int cls_of[kMaxSpecs];                  // class of every spec
    int k_lo[kMaxSpecs], k_hi[kMaxSpecs];   // inclusive sub-window, inside the plan's union window
    int mode[kMaxSpecs];                    // APX_PEAK_MAX / APX_PEAK_LOCAL_MAX
    int norm[kMaxSpecs];                    // 1 = write A / N_c
    uint32_t cls_mask[kMaxSpecs][8];        // accepted ion types of every class
};
__device__ __forceinline__ bool type_in_class(const SpecSet &ss, int cls, uint32_t t)
{
    return t == kUntyped || ((ss.cls_mask[cls][(t >> 5) & 7] >> (t & 31)) & 1u);
}

struct Plan {
    apx_plan_desc desc;            // copy (dirs pointer nulled)
    int B, D, pad, k_lo, k_hi, W;  // k_lo..k_hi = union window of all specs, W = its width
    SpecSet specs;
    float R, R2, s;
    int device;
    int path;                      // 0 = FFT kernel, 1 = MMA kernel
    int sm_count;
    int last_cuda;
    bool ingested;
    // device buffers owned by the plan
    float *d_dirs_scaled;          // [D][3]  n' = fl32(n*s)
    float2 *d_twiddle;             // [B/2]   exp(-2 pi i r / B), r < B/2   (FFT path)
    void *d_mma_table;             // twiddle operand of the windowed DFT (MMA path)
    void *d_mma_zero;              // zeros, source of the bulk copies that clear a histogram buffer (MMA path)
    float2 *d_mma_phase;           // [4][W] recombination phases of the four bin parts (MMA path)
    float *d_dirs_sorted;          // [Dp][3] scaled directions in patch order (MMA path)
    int *d_dir_perm;               // [Dp] original index of each sorted slot, -1 = padding
    int *d_dir_perm_mirror;        // [Dp] half-grid mode: index of the direction opposite to the slot's
    int Dp;                        // D rounded up to a multiple of 32
    int *d_fft_half, *d_fft_partner;   // general kernel's half-grid mode: binned member of each pair, partner of each direction
    int fft_paired;                // 1 = the general (FFT) kernel runs in half-grid mode on this plan's symmetric grid
    int mma_paired;                // 1 = half-grid mode: the grid is antipodally symmetric, one direction per pair is binned
    int tune_unit_split, tune_nacc, tune_dc;   // k_signature_mma scheduling knobs (see mma_path_prepare)
    int need_clamp;                // 1 = the bin clamp of Eq. 1 can trigger and must stay in the kernels' inner loops
    uint32_t *d_deferred;          // [0] count, [1..] material points the MMA kernel left to the FFT kernel
    int64_t cap_deferred;
    uint32_t *dbg_hist_out;        // non-null only inside apx_debug_histograms: the kernels also export their histograms
    int dbg_d0, dbg_nd;
    long long *dbg_trace;          // APX_TRACE builds only: pipeline timeline buffer of k_signature_mma (else unused)
    int dbg_trace_block, dbg_trace_cap;
    float *dbg_centre;             // [3] device copy of the debug centre
    float *dbg_sig;                // [D][2] scratch signature output of the debug run
    float *d_refine_off;           // [16] sub-cell centre offsets of apx_refine_centres
    float *d_kaxis;                // [cap_kaxis] k values of one axis of apx_fsp's reciprocal-space grid
    int cap_kaxis;
    int fsp_path;                  // 0 = tensor-core kernel (+ FP32 kernel for oversized ROIs), 1 = FP32 kernel only
    uint32_t *d_fsp_list;          // [0] count, [1..] material points k_fsp_mma left to k_fsp
    int64_t cap_fsp_list;
    uint32_t *d_type_mask;         // [8] words
    GridParams *d_grid;
    uint32_t *d_cell_start;        // [kMaxCells + 1]
    uint32_t *d_cell_cursor;       // [kMaxCells]
    uint32_t *d_scan_tiles;        // [kMaxCells / 8192] tile totals of the cell scan
    float4 *d_sorted;              // [capacity]  (x, y, z, ion type bits)
    int64_t capacity;              // ions the sorted buffers can hold
    // host staging for apx_run_host
    cudaStream_t own_stream, copy_stream;
    cudaEvent_t slab_done[2], copy_done[2];
    void *h2d_xyz, *h2d_types, *h2d_centres, *d2h_sig, *d2h_counts;   // device-side staging
    int64_t cap_xyz, cap_types, cap_centres, cap_sig, cap_counts;
};

// ---- binning arithmetic (Eq. 1 in the fp32 operation order fixed by DESIGN.md reading #15) ----------
// x = fma(n'z, dz, fma(n'y, dy, n'x*dx)); b = clamp(B/2 + floor(x), 0, B-1).
// floor via a round-down add of the magic constant 1.5*2^23 + B/2 (exact for |x| < 2^22): the low
// mantissa bits of the sum are B/2 + floor(x).  The clamp is applied on x first:
// max(x, -B/2) -> b >= 0 and min(x, B/2 - 0.25) -> b <= B-1, identical to clamping b.
__device__ __forceinline__ int bin_of(float npx, float npy, float npz, float dx, float dy, float dz,
                                      float half_b, float magic)
{
    float x = __fmaf_rn(npz, dz, __fmaf_rn(npy, dy, __fmul_rn(npx, dx)));
    x = fminf(fmaxf(x, -half_b), half_b - 0.25f);
    return __float_as_int(__fadd_rd(x, magic)) - 0x4B400000;
}
__host__ __device__ __forceinline__ float magic_for(int B) { return 12582912.0f + (float)(B / 2); }

// membership: closed ball in fp32, r2 = fma(dz,dz, fma(dy,dy, dx*dx)) <= R2
__device__ __forceinline__ bool inside(float dx, float dy, float dz, float R2)
{
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx))) <= R2;
}

// cell coordinate along one axis (monotone in v); clamped to [0, n-1]
__device__ __forceinline__ int cell_coord(float v, float o, float inv_h, int n)
{
    int c = __float2int_rd(__fmul_rn(__fsub_rn(v, o), inv_h));
    return min(max(c, 0), n - 1);
}

struct RoiCells {
    int ix0, ix1, iy0, iy1, iz0, iz1;
};

// conservative cell block of the ball around c (monotone cell_coord + a margin that covers the fp32
// rounding of p - c and of c -+ R; membership itself is always the exact fp32 test)
__device__ __forceinline__ RoiCells roi_cells(const GridParams &g, float cx, float cy, float cz, float R)
{
    RoiCells r;
    float mx = R * 1.00001f + fabsf(cx) * 1e-6f;
    float my = R * 1.00001f + fabsf(cy) * 1e-6f;
    float mz = R * 1.00001f + fabsf(cz) * 1e-6f;
    r.ix0 = cell_coord(cx - mx, g.ox, g.inv_h, g.nx); r.ix1 = cell_coord(cx + mx, g.ox, g.inv_h, g.nx);
    r.iy0 = cell_coord(cy - my, g.oy, g.inv_h, g.ny); r.iy1 = cell_coord(cy + my, g.oy, g.inv_h, g.ny);
    r.iz0 = cell_coord(cz - mz, g.oz, g.inv_h, g.nz); r.iz1 = cell_coord(cz + mz, g.oz, g.inv_h, g.nz);
    return r;
}

// launchers (each returns the cudaError_t of the launch)
cudaError_t launch_ingest(Plan *p, const float *xyz, const uint8_t *types, int64_t N, cudaStream_t st);
cudaError_t launch_signature_fft(Plan *p, const float *centres, int64_t M, float *sig, uint32_t *counts,
                                 cudaStream_t st);
// FFT kernel over a device-side list of material points (list[0] = count, list[1..] = ids)
cudaError_t launch_signature_fft_list(Plan *p, const float *centres, const uint32_t *list, int64_t M, float *sig,
                                      uint32_t *counts, cudaStream_t st);
cudaError_t launch_signature_mma(Plan *p, const float *centres, int64_t M, float *sig, uint32_t *counts,
                                 cudaStream_t st);
bool mma_path_supported(const Plan *p);
cudaError_t mma_path_prepare(Plan *p);   // builds d_mma_table
cudaError_t mma_reserve_deferred(Plan *p, int64_t need);   // deferred list of at least `need` words
cudaError_t launch_fsp_mma(Plan *p, const float *centres, int64_t M, int L, float dk, float *out, uint32_t *counts, uint32_t *list,
                           cudaStream_t st);
cudaError_t launch_fsp_mma_at(Plan *p, const float *kaxis, const float *centres, int64_t M, int L, float dk, float *out,
                              uint32_t *counts, uint32_t *list, cudaStream_t st);   // k axis at a given device address
cudaError_t mma_reserve_for(Plan *p, int64_t M);           // ... sized for any apx_query of up to M material points

}  // namespace apx

struct apx_plan : public apx::Plan {};
