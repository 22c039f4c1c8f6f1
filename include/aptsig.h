/* aptsig.h -- C ABI of libaptsig: crystallographic signatures of atom-probe point clouds on one
 * NVIDIA B200 (sm_100a).  Hot path of the real space method (RSP) of Kuehbach, Kasemer, Gault, Breen,
 * arXiv 2009.00735: for every material point (ROI centre) gather the ions of the accepted types
 * inside a sphere of radius R, project them onto every direction of a unit-sphere grid
 * (L60), histogram the signed distances into B = 2^m bins (Eq. 1; dR and f_s in the Fig. 2
 * caption, L138; one zero pad bin per side, L365), take the one-sided DFT amplitude spectrum (L73) and
 * record the highest amplitude inside a spectral bin window and its bin (L75, L416).
 *
 * Conventions
 *   - every function returns APX_OK (0) or a negative apx_status; nothing throws or aborts.
 *   - pointers marked DEVICE are CUDA device pointers on the plan's device, owned by the caller; the
 *     library never frees them and does not touch them after the stream work of the call completed.
 *     Pointers marked HOST are read (or written) before the call returns.
 *   - all work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream);
 *     calls return without synchronising unless stated.
 *   - a plan is not thread-safe; distinct plans are independent.  No global state.
 *   - there is NO CPU fallback: without a usable CUDA device apx_plan_create fails with APX_ECUDA.
 */
#ifndef APTSIG_H_
#define APTSIG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    APX_OK = 0,
    APX_EINVAL = -1,   /* bad argument: B not a power of two in 256..4096, R <= 0, D < 1, bad window, NULL */
    APX_ENOMEM = -2,   /* host or device allocation failed */
    APX_ECUDA = -3,    /* a CUDA call failed; apx_last_cuda_error() gives the cudaError_t */
    APX_ESTATE = -4,   /* apx_query / apx_debug_histograms before apx_ingest */
    APX_ERANGE = -5    /* size beyond what the plan supports (N >= 2^31, M*D >= 2^40) */
} apx_status;

/* flags */
#define APX_FLAG_FORCE_FFT 1   /* always use the general FFT kernel, even for a narrow window */
#define APX_FLAG_FORCE_MMA 2   /* fail with APX_EINVAL instead of falling back when the tensor-core
                                  windowed-DFT kernel cannot serve the plan (window too wide) */
#define APX_FLAG_NORMALISE 8   /* apx_plan_create: write A / N_c instead of A (apx_sig_spec.normalise of the one signature) */
#define APX_FLAG_LOCAL_MAX 16  /* apx_plan_create: APX_PEAK_LOCAL_MAX for the one signature (general FFT kernel) */
#define APX_FLAG_NO_PAIRING 4  /* either kernel: no half-grid mode even when the grid is antipodally
                                  symmetric (test hook; results are identical either way) */

/* peak modes (L75 "particular bins"; L149-151 "second strongest peak") */
#define APX_PEAK_MAX 0         /* highest amplitude of the window (default; L416 "the highest amplitude ... in the bin interval") */
#define APX_PEAK_LOCAL_MAX 1   /* highest LOCAL maximum of the window: bin k with A_k > A_{k-1} and A_k >= A_{k+1} (A_{B/2+1} =
                                  A_{B/2-1}); lowest k on ties; (0, k_lo) when the window has none.  The ROI-shape envelope that
                                  dominates low bins falls monotonically and is never picked.  General FFT kernel only. */
#define APX_MAX_SIGNATURES 4   /* signatures (apx_sig_spec) per plan */

typedef struct apx_plan apx_plan; /* opaque */

typedef struct {
    float R;              /* ROI radius > 0, same length unit as the coordinates (L52)                  */
    int32_t B;            /* histogram bins, power of two, 256..4096 (m = 8..12, L71)                   */
    int32_t pad;          /* 1 = paper's Eq. 1: span [-R-dR, R+dR], dR = R/(B/2-1) (L138, L365; default)
                             0 = span [-R, R] (BASELINE.json north_star wording)                         */
    int32_t k_lo, k_hi;   /* inclusive spectral-bin window, 0 <= k_lo <= k_hi <= B/2;
                             k_lo = k_hi = 0 selects [1, B/2] (every bin but DC, L122/L151)             */
    const float *dirs;    /* HOST, D x 3 direction vectors (unit vectors expected, L60), copied         */
    int32_t D;            /* number of directions, >= 1                                                  */
    uint8_t type_mask[32];/* bit t (byte t>>3, bit t&7) set = ion type t accepted (L52 "selected atom
                             types"); all 0xFF = no filter                                               */
    int32_t device;       /* CUDA device ordinal                                                         */
    int32_t flags;        /* APX_FLAG_*                                                                  */
} apx_plan_desc;

/* One signature of a multi-signature plan: "at least one [...] signature is computed from the positions of selected atom
 * types in the ROI [...] multiple signatures (for different atom types) are computed per ROI" (L52); "Signatures were
 * processed for several lattice plane families {002}, {220}, and {111}" (L208), each from "the peaks of the same bins"
 * (L214) of the amplitude spectrum. */
typedef struct {
    uint8_t type_mask[32];   /* accepted ion types, as in apx_plan_desc                                              */
    int32_t k_lo, k_hi;      /* inclusive spectral-bin window, as in apx_plan_desc (0, 0 = [1, B/2])                 */
    int32_t peak_mode;       /* APX_PEAK_MAX or APX_PEAK_LOCAL_MAX                                                   */
    int32_t normalise;       /* 1 = amplitudes are written as A / N_c (normalised intensity: ~1.0 for perfect
                                crystals, L424; 0 for an empty ROI); 0 = raw |X_k|                                    */
} apx_sig_spec;

/* Plan (step a0): derived constants R2 = fl32(R*R), s = fl32((B/2-pad)/R) = 1/dR, scaled directions
 * n' = fl32(n*s), twiddle tables; owns all internal device buffers.  *out is NULL on failure. */
int apx_plan_create(const apx_plan_desc *desc, apx_plan **out);
/* A plan that computes n_specs (1..APX_MAX_SIGNATURES) signatures per material point from ONE ingest and ONE launch:
 * ions are ingested once (union of the masks), specs with the same type mask share one gather, one binning pass and one
 * transform per direction, every spec takes its peak from its own window.  desc->type_mask / k_lo / k_hi are ignored.
 * Outputs of apx_query / apx_run / apx_run_host then hold one plane per spec, in spec order:
 *   sig float32[n_specs][M][D][2], counts uint32[n_specs][M].
 * Each plane equals what a single-signature plan with that mask and window produces. */
int apx_plan_create_multi(const apx_plan_desc *desc, const apx_sig_spec *specs, int32_t n_specs, apx_plan **out);
int apx_plan_num_signatures(const apx_plan *plan);
int apx_plan_destroy(apx_plan *plan);

/* The exact fp32 constants the kernels use (HOST out pointers, any may be NULL):
 * R2, s, and the spatial frequency of spectral bin 1, nu_1 = s/B (bin k is k*nu_1; plane spacing 1/(k nu_1)). */
int apx_plan_constants(const apx_plan *plan, float *R2, float *s, float *freq_per_bin);
/* 0 = general FFT kernel, 1 = tensor-core windowed-DFT kernel (chosen at create time from the window). */
int apx_plan_path(const apx_plan *plan);
/* 1 = half-grid mode of the plan's kernel (both kernels have one): the direction grid is antipodally symmetric (every n has its exact
 * negative in the grid, e.g. the paper's geodesic mesh, L60), so one member of every pair (n, -n) is binned and its
 * peak serves both (the histogram of -n is the mirror image: same amplitude spectrum); pairs with an ion whose
 * projection is an exact integer, where the mirror symmetry of Eq. 1's floor fails, are redone on their own.
 * 0 = every direction on its own.  Results are identical either way. */
int apx_plan_paired(const apx_plan *plan);
int apx_last_cuda_error(const apx_plan *plan);

/* Step a1: ingest an ion cloud: drop ions of rejected types and non-finite coordinates, bucket the
 * rest into a uniform cell grid (cell edge ~R/2) by a counting sort on the device.
 *   xyz   DEVICE float32[N][3]     types DEVICE uint8[N] or NULL (NULL = no type information: every
 *                                  ion is accepted, the plan's type mask is not applied)
 * The plan keeps the sorted copy (16 B per ion) until the next ingest; xyz/types are not referenced
 * after the enqueued work completed.  N = 0 is valid (all ROIs empty).  The first call with a larger N
 * than any before grows the plan's buffers (cudaMalloc: synchronises the device); apx_plan_reserve
 * sizes them ahead of time. */
int apx_ingest(apx_plan *plan, const float *xyz, const uint8_t *types, int64_t N, void *cuda_stream);

/* Steps a2-a7 for M material points against the ingested cloud.
 *   centres DEVICE float32[M][3]
 *   sig     DEVICE float32[M][D][2]: sig[m][d] = (A*, (float)k*), A* = max_{k in window} |X_k|
 *           (unnormalised, A_0 would be the ion count), k* the smallest such k.  Empty ROI: (0, k_lo).
 *   counts  DEVICE uint32[M] or NULL: number of ions in each ROI (N_c) for caller-side normalisation.
 * M = 0 is valid.  Requires a prior apx_ingest (else APX_ESTATE).  Asynchronous, except that the
 * tensor-core path grows its list of deferred material points (4 B per point and chunk) the first
 * time a larger M is seen; apx_plan_reserve avoids that. */
int apx_query(apx_plan *plan, const float *centres, int64_t M, float *sig, uint32_t *counts,
              void *cuda_stream);

/* Pre-allocate every internal buffer for clouds of up to N_max ions and queries of up to M_max material
 * points, so that later apx_ingest / apx_query / apx_run calls never allocate (and never synchronise).
 * Optional: without it buffers grow on demand. */
int apx_plan_reserve(apx_plan *plan, int64_t N_max, int64_t M_max);

/* apx_ingest followed by apx_query on the same stream (north_star's run()). */
int apx_run(apx_plan *plan, const float *xyz, const uint8_t *types, int64_t N,
            const float *centres, int64_t M, float *sig, uint32_t *counts, void *cuda_stream);

/* Same as apx_run but every array is a HOST pointer (pinned memory makes the copies asynchronous): inputs are
 * copied in on an internal stream, the material points are processed in slabs (at least four when M > 128, each
 * at most 1 GiB of signatures), and the signatures of a slab travel back on a second internal stream while the
 * next slab is computed into the other of two device staging buffers (so the device never holds more than 2 GiB
 * of output, whatever M).  Synchronises both internal streams before returning, also on errors (the end-to-end
 * entry bench.py's "e2e" figure is timed through). */
int apx_run_host(apx_plan *plan, const float *xyz, const uint8_t *types, int64_t N,
                 const float *centres, int64_t M, float *sig, uint32_t *counts);

/* Test hook: integer histograms (Eq. 1) of ONE material point for directions [d0, d0+nd):
 *   centre3 HOST float32[3],  out DEVICE uint32[nd][B] (overwritten).
 * Runs the plan's PRODUCTION kernel (the one apx_query launches for this plan: tensor-core or FFT path, with its
 * gather, packed binning arithmetic, half-grid mirroring and fix-up groups, spill / multi-pass / deferred handling)
 * on that one material point with an export switched on: the kernel copies every group's shared-memory histogram --
 * the very buffer the DFT then reads -- to `out`, decoding the tensor-core path's interleaved u16 counters; in
 * half-grid mode the direction opposite to a binned one receives the reversed histogram, as the kernel assumes. */
int apx_debug_histograms(apx_plan *plan, const float *centre3, int32_t d0, int32_t nd, uint32_t *out,
                         void *cuda_stream);

/* Step a3, host side (fp64 internally, fp32 out; `out` is HOST):
 * Fibonacci sphere: z_i = 1-(2i+1)/D, phi_i = i*pi*(3-sqrt 5)  (BASELINE.json configs 1-2). */
int apx_dirs_fibonacci(int32_t D, float *out /* D x 3 */);
/* Geodesic sphere: icosahedron subdivided `level` times (level 6 = the paper's 40 962 nodes, L60).
 * out may be NULL to query *D_out = 10*4^level + 2 only; level 0..8. */
int apx_dirs_geodesic(int32_t level, float *out, int32_t *D_out);
/* Antipodal partners of a direction grid (HOST, no GPU): partner[i] = j with dirs[j] == -dirs[i] component by
 * component (+0 and -0 are the same), or -1.  Returns 1 if every direction has a partner other than itself and no
 * direction occurs twice (the grid is antipodally symmetric: the tensor-core kernel's half-grid mode applies to it,
 * see apx_plan_paired), 0 if not, APX_EINVAL for bad arguments.  `partner` (D ints) may be NULL. */
int apx_dirs_antipodes(const float *dirs /* D x 3 */, int32_t D, int32_t *partner);

const char *apx_strerror(int status);
const char *apx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* APTSIG_H_ */
