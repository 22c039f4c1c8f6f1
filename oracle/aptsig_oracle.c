/* aptsig_oracle.c -- CPU ORACLE for the per-material-point signature of the real space method (RSP)
 * of Kuehbach, Kasemer, Gault, Breen, arXiv 2009.00735.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or constant generator with paper_2009_00735_b200/ (the CUDA path).
 *
 * It is the plain definition, written out slowly:
 *   membership : closed ball r^2 <= R^2 around the material point, optional ion-type filter
 *                ("selected atom types", L104; readings #4, #16)
 *   histogram  : Eq. 1, dR = R/(2^(m-1)-1) (Fig. 2 caption, L138), one zero pad bin
 *                on each side (L365).  With s = 1/dR = (B/2-pad)/R, Eq. 1 is b = B/2 + floor(t*s)
 *                (reading #3).  fp32 with a stated order of single-rounded operations
 *                ("single precision", L379/L403; reading #15).
 *   spectrum   : X_k = sum_j h_j exp(-2 pi i j k / B), naive O(B^2) sum in fp64, one-sided,
 *                unnormalised amplitude |X_k| (L73, L122, L151 "(unnormalised)").
 *   peak       : smallest k in [k_lo,k_hi] with maximal |X_k| (L75, L416; readings #6, #9).
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC (see oracle/build.py).
 * Every fp32 operation below is one IEEE-754 binary32 rounding; -ffp-contract=off forbids fusing.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)

static const double ORC_TWO_PI = 6.283185307179586476925286766559;

/* Step 1: R2 = fl32(R*R); s = fl32((B/2 - pad) / R) computed in fp64, rounded once. */
int orc_constants(float R, int B, int pad, float *R2, float *s)
{
    if (!(R > 0.0f) || B < 4 || (B & (B - 1)) || (pad != 0 && pad != 1)) return ORC_EINVAL;
    volatile float r2 = R * R;
    *R2 = r2;
    *s = (float)((double)(B / 2 - pad) / (double)R);
    return ORC_OK;
}

/* scaled direction n' = (fl32(nx*s), fl32(ny*s), fl32(nz*s)), one fp32 multiply each */
void orc_scale_dirs(const float *dirs, int D, float s, float *out)
{
    for (int i = 0; i < 3 * D; ++i) {
        volatile float v = dirs[i] * s;
        out[i] = v;
    }
}

static int mask_has(const uint8_t *mask32, uint8_t t) { return (mask32[t >> 3] >> (t & 7)) & 1; }

/* Step 2: brute-force membership over ALL ions (no spatial index).
 * accept iff mask[type] and fmaf(dz,dz, fmaf(dy,dy, dx*dx)) <= R2, with dx = x - cx etc.
 * Writes d = p - c (fp32) of accepted ions to rel[3*count...]; returns count (or -needed if cap too small). */
int64_t orc_members(const float *xyz, const uint8_t *types, int64_t N, const float *c, float R2,
                    const uint8_t *mask32, float *rel, int64_t cap)
{
    int64_t n = 0;
    for (int64_t i = 0; i < N; ++i) {
        if (types && !mask_has(mask32, types[i])) continue;
        float dx = xyz[3 * i + 0] - c[0];
        float dy = xyz[3 * i + 1] - c[1];
        float dz = xyz[3 * i + 2] - c[2];
        float xx = dx * dx;
        float r2 = fmaf(dz, dz, fmaf(dy, dy, xx));
        if (r2 <= R2) {
            if (n < cap) { rel[3 * n] = dx; rel[3 * n + 1] = dy; rel[3 * n + 2] = dz; }
            ++n;
        }
    }
    return n;
}

/* Step 3: Eq. 1 for one (ion, direction): x = fmaf(n'z,dz, fmaf(n'y,dy, n'x*dx)); b = B/2 + floor(x); clamp. */
static inline int orc_bin(const float *np, const float *d, int B)
{
    float xx = np[0] * d[0];
    float x = fmaf(np[2], d[2], fmaf(np[1], d[1], xx));
    int b = B / 2 + (int)floorf(x);
    if (b < 0) b = 0;
    if (b > B - 1) b = B - 1;
    return b;
}

/* histogram of `n` relative positions along one scaled direction */
void orc_hist_one(const float *rel, int64_t n, const float *nprime, int B, uint32_t *h)
{
    memset(h, 0, sizeof(uint32_t) * (size_t)B);
    for (int64_t i = 0; i < n; ++i) h[orc_bin(nprime, rel + 3 * i, B)] += 1u;
}

/* Step 4: naive one-sided DFT amplitude, fp64. theta = 2 pi ((j*k) mod B) / B. */
double orc_amp_at(const uint32_t *h, int B, int k)
{
    double re = 0.0, im = 0.0;
    for (int j = 0; j < B; ++j) {
        if (!h[j]) continue;                       /* empty bins add exactly 0 */
        double th = ORC_TWO_PI * (double)(((int64_t)j * k) % B) / (double)B;
        re += (double)h[j] * cos(th);
        im -= (double)h[j] * sin(th);
    }
    return sqrt(re * re + im * im);
}

void orc_spectrum(const uint32_t *h, int B, double *amp /* [B/2+1] */)
{
    for (int k = 0; k <= B / 2; ++k) amp[k] = orc_amp_at(h, B, k);
}

/* Histograms of one material point for directions [d0, d0+nd): out uint32[nd][B]; returns N_c.
 * `dirs` are UNIT directions float32[D][3]; scaling by s happens here (step 1). */
int64_t orc_histograms(const float *xyz, const uint8_t *types, int64_t N, const float *centre,
                       const float *dirs, int d0, int nd, float R, int B, int pad,
                       const uint8_t *mask32, uint32_t *out)
{
    float R2, s;
    if (orc_constants(R, B, pad, &R2, &s)) return ORC_EINVAL;
    int64_t n = orc_members(xyz, types, N, centre, R2, mask32, NULL, 0);
    float *rel = (float *)malloc(sizeof(float) * 3 * (size_t)(n > 0 ? n : 1));
    if (!rel) return ORC_ENOMEM;
    orc_members(xyz, types, N, centre, R2, mask32, rel, n);
    for (int d = 0; d < nd; ++d) {
        float np[3];
        orc_scale_dirs(dirs + 3 * (size_t)(d0 + d), 1, s, np);
        orc_hist_one(rel, n, np, B, out + (size_t)d * B);
    }
    free(rel);
    return n;
}

/* Steps 1-5 for M material points x D directions.
 *   sig    float32[M][D][2] = ((float)A_k*, (float)k*),   counts uint32[M] (may be NULL)
 *   winamp double[M][D][k_hi-k_lo+1] (may be NULL): all window amplitudes, for the tie rule in tests
 * The inner sum is orc_amp_at's sum with cos/sin of the same argument 2 pi r / B read from a table
 * built by the same expression (so the values are bit-identical to orc_amp_at).
 * Threads: OpenMP over material points (nthreads <= 0: all cores).  Returns 0 or a negative error. */
int orc_signatures(const float *xyz, const uint8_t *types, int64_t N,
                   const float *centres, int64_t M, const float *dirs, int D,
                   float R, int B, int pad, int k_lo, int k_hi, const uint8_t *mask32,
                   float *sig, uint32_t *counts, double *winamp, int nthreads)
{
    float R2, s;
    if (orc_constants(R, B, pad, &R2, &s)) return ORC_EINVAL;
    if (k_lo == 0 && k_hi == 0) { k_lo = 1; k_hi = B / 2; }
    if (k_lo < 0 || k_hi > B / 2 || k_lo > k_hi || D < 0 || M < 0) return ORC_EINVAL;
    const int W = k_hi - k_lo + 1;
    double *ct = (double *)malloc(sizeof(double) * 2 * (size_t)B);
    float *nps = (float *)malloc(sizeof(float) * 3 * (size_t)(D > 0 ? D : 1));
    if (!ct || !nps) { free(ct); free(nps); return ORC_ENOMEM; }
    double *st = ct + B;
    for (int r = 0; r < B; ++r) {
        double th = ORC_TWO_PI * (double)r / (double)B;
        ct[r] = cos(th);
        st[r] = sin(th);
    }
    orc_scale_dirs(dirs, D, s, nps);
    int err = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t m = 0; m < M; ++m) {
        const float *c = centres + 3 * m;
        int64_t n = orc_members(xyz, types, N, c, R2, mask32, NULL, 0);
        float *rel = (float *)malloc(sizeof(float) * 3 * (size_t)(n > 0 ? n : 1));
        uint32_t *h = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)B);
        if (!rel || !h) { err = ORC_ENOMEM; free(rel); free(h); continue; }
        orc_members(xyz, types, N, c, R2, mask32, rel, n);
        if (counts) counts[m] = (uint32_t)n;
        for (int d = 0; d < D; ++d) {
            orc_hist_one(rel, n, nps + 3 * (size_t)d, B, h);
            double best = -1.0;
            int kbest = k_lo;
            for (int k = k_lo; k <= k_hi; ++k) {
                double re = 0.0, im = 0.0;
                for (int j = 0; j < B; ++j) {
                    if (!h[j]) continue;
                    int r = (int)(((int64_t)j * k) % B);
                    re += (double)h[j] * ct[r];
                    im -= (double)h[j] * st[r];
                }
                double a = sqrt(re * re + im * im);
                if (winamp) winamp[((size_t)m * D + d) * W + (k - k_lo)] = a;
                if (a > best) { best = a; kbest = k; }      /* strict >: lowest k wins ties */
            }
            sig[((size_t)m * D + d) * 2 + 0] = (float)best;
            sig[((size_t)m * D + d) * 2 + 1] = (float)kbest;
        }
        free(rel);
        free(h);
    }
    free(ct);
    free(nps);
    return err;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
