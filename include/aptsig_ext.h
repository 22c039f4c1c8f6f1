/* aptsig_ext.h -- C ABI of the steps that follow the signature computation in the paper's workflow:
 *   NEXT-4  adaptive refinement of the ROI grid
 *   NEXT-1  indexing of signatures against rotated references, Eq. 3 (L98, L369-373, L395, L416)
 *   NEXT-3  reciprocal space method (FSP), Eq. 2 (L79-84, L389-393)
 * Same conventions as aptsig.h (status codes, DEVICE / HOST pointers, `cuda_stream`, no CPU fallback).
 */
#ifndef APTSIG_EXT_H_
#define APTSIG_EXT_H_

#include "aptsig.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ---------------------------------------------------------------------------------------------------------------
 * NEXT-4: grid refinement.  "The distribution of signature intensity values for each signature and every ROI is analysed
 * to identify those positions where the maximum intensity per signature exceeds a threshold value (here choosing
 * kappa >= 0.75 normalised image intensity).  In a second iteration [...] splitting the corresponding ROI grid cell into
 * 5^3 cells and placing that amount of new ROIs at the respective centre" (L210).
 * Normalised intensity = A / N_c (amplitude over the ROI's ion count; L424: ~1.0 for perfect crystals); empty ROI = 0. */

/* kappa_max[m] = max_d sig[m][d][0] / counts[m].
 *   sig DEVICE float32[M][D][2] (as written by apx_query; D = the plan's),  counts DEVICE uint32[M],
 *   kappa_max DEVICE float32[M] (out). */
int apx_intensity_max(apx_plan *plan, const float *sig, const uint32_t *counts, int64_t M, float *kappa_max,
                      void *cuda_stream);

/* Ordered stream compaction: selected[0 .. *n_selected) = the m, ascending, with kappa_max[m] >= kappa.
 *   selected DEVICE uint32[M] (out),  n_selected DEVICE uint32[1] (out).  M < 2^31. */
int apx_refine_select(apx_plan *plan, const float *kappa_max, int64_t M, float kappa, uint32_t *selected,
                      uint32_t *n_selected, void *cuda_stream);

/* New ROI centres: for the s-th selected material point m, split^3 centres
 *   c' = fl32(c_m + fl32(((i + 0.5)/split - 0.5) * spacing)) per axis (i = 0..split-1; offsets computed in fp64 and
 *   rounded once), written to out[(s*split^3 + (iz*split + iy)*split + ix)][3].
 *   centres DEVICE float32[M][3], selected / n_selected as written by apx_refine_select (the count is read on the
 *   device: no host synchronisation), out DEVICE float32[max_selected * split^3][3]; selected points beyond
 *   max_selected are dropped.  1 <= split <= 16. */
int apx_refine_centres(apx_plan *plan, const float *centres, const uint32_t *selected, const uint32_t *n_selected,
                       int64_t max_selected, float spacing, int32_t split, float *out, void *cuda_stream);

/* ---------------------------------------------------------------------------------------------------------------
 * NEXT-1: indexing.  "First, the intensities [...] are normalised individually.  Second, a user-defined sub-set of the FE
 * nodes is defined (here N_v^ = 1000) for each reference.  We pick those nodes for which the signal is strongest.  Third,
 * orientation set G is used to rotate each of the N_v^ FE nodes and compute its closest neighbouring node p^g_{v,c}"
 * (L369); Delta^g_c = sum_v (S^msr_c|p^g_{v,c} - S^g_c|v)^2 (Eq. 3).  One indexer = one crystal structure candidate. */
#define APX_INDEX_MAX_K 8      /* best solutions kept per material point (the paper inspected up to 1000, L416) */

typedef struct apx_indexer apx_indexer; /* opaque */

/* Pre-processing (synchronises the device): strongest nodes of the reference and the look-up table on the device.
 *   dirs      HOST float32[D][3]   the mesh nodes' unit normals (the plan's direction grid)
 *   quats     HOST float32[Ng][4]  orientation set, unit quaternions (w, x, y, z), active rotations v' = q v q*
 *   ref_image HOST float32[D]      NORMALISED reference intensities of this candidate (e.g. apx_query amplitudes of a
 *                                  synthetic single crystal divided by its counts)
 *   n_hat     number of strongest nodes compared (1 <= n_hat <= D) */
int apx_indexer_create(const float *dirs, int32_t D, const float *quats, int64_t Ng, const float *ref_image,
                       int32_t n_hat, int32_t device, apx_indexer **out);
int apx_indexer_destroy(apx_indexer *ix);
/* The chosen nodes, strongest first (HOST int32[n_hat]) and their reference intensities (HOST float32[n_hat]). */
int apx_indexer_nodes(const apx_indexer *ix, int32_t *nodes, float *ref_values);
/* Rows [g0, g0+ng) of the look-up table copied to HOST int32[ng][n_hat] (synchronises). */
int apx_indexer_lut(apx_indexer *ix, int64_t g0, int64_t ng, int32_t *out);
int apx_last_cuda_error_indexer(const apx_indexer *ix);

/* Eq. 3 for M measured signatures against every orientation; the K smallest image differences per material point.
 *   sig        DEVICE float32[M][D][2]  as written by apx_query (amplitude at [..][0])
 *   counts     DEVICE uint32[M], or NULL when sig already holds normalised intensities
 *   best_delta DEVICE float32[M][K] (out)  ascending;  best_g DEVICE int32[M][K] (out)  orientation indices, the lower
 *              index first among equal Delta.  1 <= K <= APX_INDEX_MAX_K. */
int apx_index(apx_indexer *ix, const float *sig, const uint32_t *counts, int64_t M, int32_t K, float *best_delta,
              int32_t *best_g, void *cuda_stream);

/* Host-side orientation set standing in for the paper's MTEX grid (L367; not in the container): cubic lattice of
 * Rodrigues vectors (lattice constant tan(spacing/2), origin = identity) cut to the m-3m fundamental zone
 * |r_i| <= sqrt2 - 1, |r_1|+|r_2|+|r_3| <= 1; quaternions (w > 0) in lattice order (z, y, x).
 * quats may be NULL to query *Ng only; HOST float32[*Ng][4]. */
int apx_so3_grid_cubic(float spacing_deg, float *quats, int64_t *Ng);

/* ---------------------------------------------------------------------------------------------------------------
 * NEXT-3: reciprocal space method (FSP).  "evaluate Eq. 2 to compute a direct Fourier transform of the positions for all
 * atoms N_w of a selected atom type within each ROI c": F(k) = sum_w exp(-2 i pi k.(p_w - p_c)) (Eq. 2), on a cubic
 * grid of L_D^3 reciprocal-space positions (L389: L_D = 64..512, "k in [-2pi, +2pi]^3"); the signature is a 3-D image stack.
 * Here: k = (kx[ix], ky[iy], kz[iz]), each axis L points uniformly spaced over [-k_max, +k_max] (both ends included;
 * computed in fp64, rounded once to fp32), in units of 1/length of the coordinates (the 2 pi is in the exponent, as printed).
 *   centres DEVICE float32[M][3];  out DEVICE float32[M][L][L][L], out[m][iz][iy][ix] = |F(k)|;
 *   counts DEVICE uint32[M] or NULL (N_w per ROI).  Uses the plan's R, ion-type filter and ingested cloud (APX_ESTATE
 *   without apx_ingest).  1 <= L <= 1024, M * L * ceil(L/64)^2 < 2^31. */
int apx_fsp(apx_plan *plan, const float *centres, int64_t M, float k_max, int32_t L, float *out, uint32_t *counts,
            void *cuda_stream);
/* Kernel choice of apx_fsp: 0 (default) = the tensor-core kernel (Eq. 2 per z-slice pair as one real GEMM of fp16 hi + lo
 * split operands, fp32 accumulation in TMEM), with the FP32 kernel serving ROIs of more than 2560 ions in the same stream;
 * 1 = the FP32-pipe kernel for everything.  Results agree within the tolerance derived in DESIGN.md section 2. */
int apx_fsp_set_path(apx_plan *plan, int32_t path);

/* apx_fsp for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same operation (Eq. 2), the same kernels, arguments, layout and results as apx_fsp with the
 * plan's current apx_fsp_set_path choice, but the scratch apx_fsp keeps in lazily (re)allocated plan buffers -- the k axis
 * (float32[L]) and the device list of ROIs the tensor-core kernel hands to the FP32 kernel (uint32[1 + M]) -- lives in ONE
 * file-scope `static __device__` array of APX_FSP_NOALLOC_SCRATCH_BYTES inside the library (held by every GPU that loads
 * the library until the process exits).  The call performs no cudaMalloc / cudaFree / allocating library routine and no
 * host-to-device copy: the k axis is computed on the device (same fp64 formula, rounded once) and the list count is
 * cleared by a small kernel in `cuda_stream` ahead of the FSP kernels.
 *   Limits: M <= APX_FSP_NOALLOC_MAX_M and L <= APX_FSP_NOALLOC_MAX_L, else APX_ERANGE and nothing is launched
 *   (apx_fsp_noalloc_limits reports the numbers); all other argument rules and status codes are apx_fsp's.
 *   Sharing: every call on a device uses the same array, which keeps the last call's contents.  Calls in one stream are
 *   ordered and safe; calls that overlap on the GPU (different streams, or several plans on one device) RACE on it --
 *   serialise them, or use apx_fsp.
 *   The first call on a device resolves the array's device address (cudaGetSymbolAddress, once per device); make that
 *   first call outside stream capture. */
#define APX_FSP_NOALLOC_MAX_M 16384
#define APX_FSP_NOALLOC_MAX_L 1024
#define APX_FSP_NOALLOC_SCRATCH_BYTES 69888   /* 4096 (k axis) + 65792 (list: 1 + 16384 words, padded to 256 B) */
int apx_fsp_noalloc(apx_plan *plan, const float *centres, int64_t M, float k_max, int32_t L, float *out, uint32_t *counts,
                    void *cuda_stream);
/* The limits above, for bindings: any pointer may be NULL.  Returns APX_OK. */
int apx_fsp_noalloc_limits(int64_t *max_M, int32_t *max_L, int64_t *scratch_bytes);

#ifdef __cplusplus
}
#endif
#endif /* APTSIG_EXT_H_ */
