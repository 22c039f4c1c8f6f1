// signature_fft.cu -- general signature kernel (any window, B = 256..4096): steps a2, a4-a7.
//
// One CTA (16 warps) = one material point x a chunk of direction groups; a group = G directions
// (G = 32 for B <= 1024, 16 for B = 2048, 8 for B = 4096: B*G*4 bytes = at most 128 KB of shared memory).
//   gather   : the ROI's ions are collected once per CTA into shared memory (packed dx, dy, dz).
//   binning  : lane = direction (lane % G), the warps split the ions; counter of (bin b, direction d) is the
//              32-bit word b*G + d, so for G = 32 every lane of a shared atomic hits its own bank (Eq. 1,
//              PAPER.md L68-71).  A pair costs FMUL, 2 FFMA, FADD.RM, IMAD, ATOMS.
//   FFT      : the B counts of a direction are read as N = B/2 complex points z_j = (h_2j, h_2j+1) (real input
//              packing; the paper calls a real-to-complex library FFT per histogram, L73/L379) and transformed
//              in place by radix-8 decimation-in-frequency passes held in registers (plus one radix-2/4 pass):
//              512/G threads per direction, each butterfly reads and writes only its own lane's bank.  The first
//              pass converts the integer counts to float on load.
//   peak     : the split step X_k = (Z_k + conj Z_{N-k})/2 - i w^k (Z_k - conj Z_{N-k})/2 is evaluated only for
//              the window bins, |X_k|^2 arg-max with the lowest k on ties (L75, L416), one sqrt at the end.
// Histograms and spectra never leave the SM.  ROIs with more ions than the shared buffer holds are binned by
// streaming their cell rows from global memory again for every group (no size limit).
#include "common.cuh"

namespace apx {

constexpr int kFftThreads = 512;
constexpr int kFftWarps = kFftThreads / 32;

struct FftParams {
    const float4 *sorted;
    const uint32_t *cell_start;
    const GridParams *grid;
    const float *centres;
    const float *dirs_scaled;
    const float2 *tw;          // [B/2] exp(-2 pi i r / B)
    float2 *sig;
    uint32_t *counts;
    const uint32_t *list;      // nullptr = direct mode; else list[0] = count, list[1..] = material point ids
    uint32_t *hist_out;        // test hook (apx_debug_histograms, M = 1): uint32[hist_nd][B] histograms of the directions
    int hist_d0, hist_nd;      // [hist_d0, hist_d0 + hist_nd), copied from the shared counters the FFT is about to read
    // half-grid mode (antipodally symmetric grids, see the kernel): half[u] = the member of pair u that is binned,
    // partner[d] = index of -d; nullptr = every direction on its own
    const int *half, *partner;
    int Dh;                    // pairs (D / 2)
    int D, k_lo, k_hi, cap, nchunks, ngroups, clamp;
    float R, R2;
    SpecSet ss;                // signatures of the plan: classes (type masks) and per-spec windows / modes
    int64_t M;                 // material points of the call: plane stride of sig (M * D) and counts (M)
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }          // a * (-i)

// w_B^r for 0 <= r < B from the half table (w^{r + B/2} = -w^r)
template <int B>
__device__ __forceinline__ float2 twiddle(const float2 *tw, int r)
{
    const float2 w = tw[r & (B / 2 - 1)];
    return (r & (B / 2)) ? make_float2(-w.x, -w.y) : w;
}

// forward DFT of R points in registers (R = 2, 4, 8), natural order in, natural order out
template <int R>
__device__ __forceinline__ void dft(float2 (&x)[R])
{
    if (R == 2) {
        const float2 a = x[0], b = x[1];
        x[0] = cadd(a, b); x[1] = csub(a, b);
    } else if (R == 4) {
        const float2 a = cadd(x[0], x[2]), b = csub(x[0], x[2]), c = cadd(x[1], x[3]), d = mul_mi(csub(x[1], x[3]));
        x[0] = cadd(a, c); x[2] = csub(a, c); x[1] = cadd(b, d); x[3] = csub(b, d);
    } else {
        const float h = 0.70710678118654752440f;
        // stage 1: pairs (m, m+4)
        float2 a0 = cadd(x[0], x[4]), a1 = cadd(x[1], x[5]), a2 = cadd(x[2], x[6]), a3 = cadd(x[3], x[7]);
        float2 b0 = csub(x[0], x[4]), b1 = csub(x[1], x[5]), b2 = csub(x[2], x[6]), b3 = csub(x[3], x[7]);
        // twiddles w_8^m on the odd half: 1, (1-i)/sqrt2, -i, (-1-i)/sqrt2
        b1 = make_float2(h * (b1.x + b1.y), h * (b1.y - b1.x));
        b2 = mul_mi(b2);
        b3 = make_float2(h * (b3.y - b3.x), -h * (b3.x + b3.y));
        // two 4-point DFTs: even outputs from a, odd outputs from b
        float2 c0 = cadd(a0, a2), c1 = csub(a0, a2), c2 = cadd(a1, a3), c3 = mul_mi(csub(a1, a3));
        x[0] = cadd(c0, c2); x[4] = csub(c0, c2); x[2] = cadd(c1, c3); x[6] = csub(c1, c3);
        float2 d0 = cadd(b0, b2), d1 = csub(b0, b2), d2 = cadd(b1, b3), d3 = mul_mi(csub(b1, b3));
        x[1] = cadd(d0, d2); x[5] = csub(d0, d2); x[3] = cadd(d1, d3); x[7] = csub(d1, d3);
    }
}

// One in-place decimation-in-frequency pass of radix R over sub-transforms of length L (N = B/2 points per
// direction, T threads per direction, this thread = t).  Element e of direction d: re at word (2e)*G + d,
// im at (2e+1)*G + d.  kFirst: the buffer still holds the integer counts.
template <int B, int G, int R, bool kFirst>
__device__ __forceinline__ void fft_pass(float *buf, const float2 *tw, int d, int t, int L)
{
    constexpr int N = B / 2, T = kFftThreads / G;
    const int span = L / R;                                    // distance between the R inputs of a butterfly
    for (int bi = t; bi < N / R; bi += T) {
        const int j = bi & (span - 1), base = (bi - j) * R + j;  // block start + j
        float2 x[R];
#pragma unroll
        for (int m = 0; m < R; ++m) {
            const int e = base + m * span;
            if (kFirst) {
                const uint32_t *ub = reinterpret_cast<const uint32_t *>(buf);
                x[m] = make_float2((float)ub[(2 * e) * G + d], (float)ub[(2 * e + 1) * G + d]);
            } else {
                x[m] = make_float2(buf[(2 * e) * G + d], buf[(2 * e + 1) * G + d]);
            }
        }
        dft<R>(x);
        const int tstep = j * (B / L);                          // w_L^{j q} = w_B^{j q B / L}
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const float2 y = (q == 0 || L == R) ? x[q] : cmul(x[q], twiddle<B>(tw, tstep * q));
            const int e = base + q * span;
            buf[(2 * e) * G + d] = y.x;
            buf[(2 * e + 1) * G + d] = y.y;
        }
    }
}

// position of frequency k after the passes (radices 8, 8[, 8][, 2|4]): digit reversal in mixed radix
template <int B>
__device__ __forceinline__ int fft_pos(int k)
{
    constexpr int N = B / 2;
    constexpr int kP8 = (N >= 512) ? 3 : 2;
    int rem = N, pos = 0;
#pragma unroll
    for (int p = 0; p < kP8; ++p) {
        rem >>= 3;
        pos += (k & 7) * rem;
        k >>= 3;
    }
    return pos + k;                                             // last digit (radix rem = 1, 2 or 4) has weight 1
}

// Gather (step a2): every warp walks x-rows of cells (contiguous in the sorted array), keeps ions with
// r^2 <= R2 and appends d = p - c as a packed 12-byte record.  *s_n may exceed cap (then the streaming path is used).
__device__ __forceinline__ void gather_roi(const FftParams &p, const GridParams &g, const RoiCells &rc,
                                           float cx, float cy, float cz, float *ions, int *s_n, int cls)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
    for (int row = wid; row < ny_r * nz_r; row += kFftWarps) {
        int iy = rc.iy0 + row % ny_r, iz = rc.iz0 + row / ny_r;
        int base = (iz * g.ny + iy) * g.nx;
        uint32_t beg = p.cell_start[base + rc.ix0], end = p.cell_start[base + rc.ix1 + 1];
        for (uint32_t i = beg + lane; i < ((end - beg + 31u) & ~31u) + beg; i += 32) {
            bool in = false;
            float dx = 0.f, dy = 0.f, dz = 0.f;
            if (i < end) {
                float4 q = p.sorted[i];
                dx = __fsub_rn(q.x, cx); dy = __fsub_rn(q.y, cy); dz = __fsub_rn(q.z, cz);
                in = inside(dx, dy, dz, p.R2) && (p.ss.n_classes == 1 || type_in_class(p.ss, cls, __float_as_uint(q.w)));
            }
            unsigned msk = __ballot_sync(0xffffffffu, in);
            if (msk) {
                int pos = 0;
                if (lane == 0) pos = atomicAdd(s_n, __popc(msk));
                pos = __shfl_sync(0xffffffffu, pos, 0) + __popc(msk & ((1u << lane) - 1u));
                if (in && pos < p.cap) { ions[3 * pos] = dx; ions[3 * pos + 1] = dy; ions[3 * pos + 2] = dz; }
            }
        }
    }
}

template <int B, bool kHalf>
__global__ void __launch_bounds__(kFftThreads, 1) k_signature_fft(const __grid_constant__ FftParams p)
{
    constexpr int G = (B <= 1024) ? 32 : 32768 / B;            // directions per group
    constexpr int N = B / 2, T = kFftThreads / G, LPD = 32 / G; // threads per direction, ions per warp instruction
    constexpr int kP8 = (N >= 512) ? 3 : 2;                    // radix-8 passes
    constexpr int kLast = N >> (3 * kP8);                      // remaining radix: 1, 2 or 4
    extern __shared__ __align__(16) unsigned char smem[];
    float *buf = reinterpret_cast<float *>(smem);                                  // [B][G] counts, then the transform
    float2 *s_tw = reinterpret_cast<float2 *>(buf + (size_t)B * G);                // [B/2]
    float2 *cand = s_tw + B / 2;                                                   // [T][G]
    float *ions = reinterpret_cast<float *>(cand + T * G);                         // [cap][3]
    __shared__ int s_n, s_nfix;
    __shared__ uint32_t s_mask;
    __shared__ int s_fix[2 * G];
    // Half-grid mode.  For -n every product and sum of Eq. 1's projection is negated exactly, so b(-n) = B - 1 - b(n) unless
    // the projection is an exact integer: the histogram of -n is the mirror image of that of n and has the same amplitude
    // spectrum.  A group then holds one member of G pairs and writes each peak to both directions.  Pairs that met an
    // exact-integer projection (RD(x + magic) = RU(x + magic)) are flagged in s_mask; their -n members are collected in
    // s_fix and binned on their own, G at a time, in fix-up groups between the ordinary ones (the list never holds more than
    // 2G - 1 entries).  Results are identical to the full grid.
    constexpr bool halfmode = kHalf;                            // (p.half != nullptr)
    const int units = halfmode ? p.Dh : p.D;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d = lane % G, t = warp * LPD + lane / G;                             // direction slot, thread index within it
    for (int i = tid; i < B / 2; i += kFftThreads) s_tw[i] = p.tw[i];
    const GridParams g = *p.grid;
    const float half_b = (float)(B / 2), magic = magic_for(B);

    // direct mode: one (material point, chunk) per CTA.  list mode: a persistent grid walks the items of the
    // material points named in list[1 .. list[0]].
    const int64_t n_items = p.list ? (int64_t)p.list[0] * p.nchunks : (int64_t)gridDim.x;
    for (int64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int64_t m = p.list ? (int64_t)p.list[1 + item / p.nchunks] : item / p.nchunks;
        const int chunk = (int)(item % p.nchunks);
        const int g_begin = (int)((int64_t)chunk * p.ngroups / p.nchunks);
        const int g_end = (int)((int64_t)(chunk + 1) * p.ngroups / p.nchunks);
        const float cx = p.centres[3 * m], cy = p.centres[3 * m + 1], cz = p.centres[3 * m + 2];
        const RoiCells rc = roi_cells(g, cx, cy, cz, p.R);

      for (int cls = 0; cls < p.ss.n_classes; ++cls) {     // specs with the same type mask share gather, binning and FFT
        __syncthreads();                 // previous item done with the shared buffers; s_tw loaded
        if (tid == 0) { s_n = 0; s_nfix = 0; }
        __syncthreads();
        if (g.n_accepted) gather_roi(p, g, rc, cx, cy, cz, ions, &s_n, cls);
        __syncthreads();
        const int n = s_n;
        if (chunk == 0 && tid == 0 && p.counts)
            for (int sp = 0; sp < p.ss.n_specs; ++sp)
                if (p.ss.cls_of[sp] == cls) p.counts[(size_t)sp * p.M + m] = (uint32_t)n;
        const bool stream = n > p.cap;
        if (n == 0 && !p.hist_out) {
            // empty ROI: all counters stay zero -> amplitude 0, lowest bin of each window (also for the local-maximum mode: no bin
            // is a local maximum, the initial candidate k_lo stands); written without binning or transforming anything
            for (int u = g_begin * G + tid; u < min(g_end * G, units); u += kFftThreads) {
                const int dsel = halfmode ? p.half[u] : u, dpart = halfmode ? p.partner[dsel] : -1;
                for (int sp = 0; sp < p.ss.n_specs; ++sp) {
                    if (p.ss.cls_of[sp] != cls) continue;
                    float2 *out = p.sig + (size_t)sp * p.M * p.D + (size_t)m * p.D;
                    const float2 res = make_float2(0.0f, (float)p.ss.k_lo[sp]);
                    out[dsel] = res;
                    if (dpart >= 0) out[dpart] = res;
                }
            }
            continue;
        }

        for (int gi = g_begin;;) {
            // ordinary group gi, or -- half-grid mode -- a fix-up group as soon as G flagged partners wait (all of them once the
            // ordinary groups are done).  s_nfix was last written before the barrier that ended the previous iteration.
            const int nf = halfmode ? s_nfix : 0;
            const bool fix = nf >= G || (gi >= g_end && nf > 0);
            if (!fix && gi >= g_end) break;
            const int fcnt = fix ? min(nf, G) : 0;
            int dsel = -1, dpart = -1;                          // direction of this lane's slot, its partner (written too)
            if (!fix) {
                const int u = gi * G + d;
                if (u < units) { dsel = halfmode ? p.half[u] : u; dpart = halfmode ? p.partner[dsel] : -1; }
            } else if (d < fcnt) {
                dsel = s_fix[nf - fcnt + d];
            }
            const bool detect = halfmode && !fix;
            if (tid == 0) s_mask = 0u;                          // (the previous iteration's readers are behind its last barrier)
            // ---- clear the counters -----------------------------------------------------------------
            {
                uint4 *h = reinterpret_cast<uint4 *>(buf);
                for (int i = tid; i < B * G / 4; i += kFftThreads) h[i] = make_uint4(0, 0, 0, 0);
            }
            __syncthreads();
            if (tid == 0 && fix) s_nfix = nf - fcnt;            // (every thread has read nf and its list entry)
            // ---- project-and-bin (step a4): lane = direction, the T threads of a direction split the ions --
            {
                const int dg = max(dsel, 0);
                bool flagged = false;                           // this thread met an exact-integer projection
                const float npx = p.dirs_scaled[3 * dg], npy = p.dirs_scaled[3 * dg + 1], npz = p.dirs_scaled[3 * dg + 2];
                // bin of one ion (Eq. 1, clamped like bin_of); notes an exact-integer projection in half-grid mode
                auto bin_x = [&](float dx, float dy, float dz) -> int {
                    float x = __fmaf_rn(npz, dz, __fmaf_rn(npy, dy, __fmul_rn(npx, dx)));
                    x = fminf(fmaxf(x, -half_b), half_b - 0.25f);
                    const uint32_t ua = __float_as_uint(__fadd_rd(x, magic));
                    if (detect) flagged |= ua == __float_as_uint(__fadd_ru(x, magic));
                    return (int)(ua - 0x4B400000u);
                };
                uint32_t *cnt = reinterpret_cast<uint32_t *>(buf) + d;
                if (!stream) {
                    // thread t takes ions t, t+T, ...; four independent chains per iteration
                    const uint32_t cb = (uint32_t)__cvta_generic_to_shared(cnt) - 0x4B400000u * (uint32_t)(4 * G);
                    int i = t;
                    for (; i + 3 * T < n; i += 4 * T) {
                        float3 q[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) q[u] = make_float3(ions[3 * (i + u * T)], ions[3 * (i + u * T) + 1], ions[3 * (i + u * T) + 2]);
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            float x = __fmaf_rn(npz, q[u].z, __fmaf_rn(npy, q[u].y, __fmul_rn(npx, q[u].x)));
                            if (p.clamp) x = fminf(fmaxf(x, -half_b), half_b - 0.25f);
                            const uint32_t ua = __float_as_uint(__fadd_rd(x, magic));
                            if (detect) flagged |= ua == __float_as_uint(__fadd_ru(x, magic));
                            asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(ua * (uint32_t)(4 * G) + cb), "r"(1u) : "memory");
                        }
                    }
                    for (; i < n; i += T)
                        atomicAdd(cnt + bin_x(ions[3 * i], ions[3 * i + 1], ions[3 * i + 2]) * G, 1u);
                } else {
                    // ROI larger than the shared ion buffer: walk the cell rows again, one ion per (warp, lane / G)
                    const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
                    for (int row = warp; row < ny_r * nz_r; row += kFftWarps) {
                        const int iy = rc.iy0 + row % ny_r, iz = rc.iz0 + row / ny_r;
                        const int base = (iz * g.ny + iy) * g.nx;
                        const uint32_t beg = p.cell_start[base + rc.ix0], end = p.cell_start[base + rc.ix1 + 1];
                        for (uint32_t i = beg + lane / G; i < end; i += LPD) {
                            const float4 q = p.sorted[i];
                            const float dx = __fsub_rn(q.x, cx), dy = __fsub_rn(q.y, cy), dz = __fsub_rn(q.z, cz);
                            if (inside(dx, dy, dz, p.R2) && (p.ss.n_classes == 1 || type_in_class(p.ss, cls, __float_as_uint(q.w))))
                                atomicAdd(cnt + bin_x(dx, dy, dz) * G, 1u);
                        }
                    }
                }
                if (flagged) atomicOr(&s_mask, 1u << d);
            }
            __syncthreads();
            if (p.hist_out && cls == 0) {                        // test hook (first class): counters complete, FFT not started
                const uint32_t *ub = reinterpret_cast<const uint32_t *>(buf);
                for (int i = tid; i < B * G; i += kFftThreads) {
                    const int b = i / G, dg = gi * G + i % G;
                    if (dg < p.D && dg >= p.hist_d0 && dg < p.hist_d0 + p.hist_nd)
                        p.hist_out[(size_t)(dg - p.hist_d0) * B + b] = ub[i];
                }
                __syncthreads();
            }
            // ---- packed real FFT (step a5): radix-8 DIF passes in place, then the remaining radix 2 / 4 ----
            fft_pass<B, G, 8, true>(buf, s_tw, d, t, N);
            __syncthreads();
            fft_pass<B, G, 8, false>(buf, s_tw, d, t, N / 8);
            __syncthreads();
            if (kP8 == 3) {
                fft_pass<B, G, 8, false>(buf, s_tw, d, t, N / 64);
                __syncthreads();
            }
            if (kLast > 1) {
                fft_pass<B, G, (kLast > 1 ? kLast : 2), false>(buf, s_tw, d, t, kLast);
                __syncthreads();
            }
            // ---- split step on the window + arg-max (steps a5 tail, a6), once per spec of this class ---------------
            // 4 |X_k|^2 of spectral bin k (0 <= k <= B/2 + 1; A_{B/2+1} = A_{B/2-1} by conjugate symmetry)
            auto power_at = [&](int k) -> float {
                if (k > N) k = B - k;
                const int ea = fft_pos<B>(k & (N - 1)), eb = fft_pos<B>((N - k) & (N - 1));
                const float2 za = make_float2(buf[(2 * ea) * G + d], buf[(2 * ea + 1) * G + d]);
                const float2 zb = make_float2(buf[(2 * eb) * G + d], buf[(2 * eb + 1) * G + d]);
                const float2 w = (k < N) ? s_tw[k] : make_float2(-1.0f, 0.0f);
                const float er = za.x + zb.x, ei = za.y - zb.y;          // Z_k + conj Z_{N-k}
                const float orr = za.x - zb.x, oi = za.y + zb.y;         // Z_k - conj Z_{N-k}
                // -i * w * (orr + i oi) = (w.y*orr + w.x*oi) + i (w.y*oi - w.x*orr)
                const float xr = er + (w.y * orr + w.x * oi);
                const float xi = ei + (w.y * oi - w.x * orr);
                return xr * xr + xi * xi;
            };
            // flagged pairs: the -n member goes to the fix-up list (published by the barriers of the spec loop below)
            if (detect && tid < G && dpart >= 0 && ((s_mask >> tid) & 1u)) s_fix[atomicAdd(&s_nfix, 1)] = dpart;
            for (int sp = 0; sp < p.ss.n_specs; ++sp) {
                if (p.ss.cls_of[sp] != cls) continue;
                const int s_lo = p.ss.k_lo[sp], s_hi = p.ss.k_hi[sp];
                const bool local = p.ss.mode[sp] == APX_PEAK_LOCAL_MAX;
                float best = -1.0f;
                int kbest = s_lo;
                for (int k = s_lo + t; k <= s_hi; k += T) {
                    const float pw = power_at(k);
                    // local-maximum mode (reading #20): only bins with A_k > A_{k-1} and A_k >= A_{k+1} compete
                    if (local && !(pw > power_at(k == 0 ? 1 : k - 1) && pw >= power_at(k + 1))) continue;
                    if (pw > best) { best = pw; kbest = k; }              // ascending k per thread: lowest k kept on ties
                }
                cand[t * G + d] = make_float2(best, __int_as_float(kbest));
                __syncthreads();
                if (tid < G) {
                    float bb = -1.0f;
                    int kb = s_lo;
                    for (int s = 0; s < T; ++s) {
                        const float2 c = cand[s * G + tid];
                        const int ck = __float_as_int(c.y);
                        if (c.x > bb || (c.x == bb && ck < kb)) { bb = c.x; kb = ck; }
                    }
                    float amp = 0.5f * sqrtf(fmaxf(bb, 0.0f));
                    if (p.ss.norm[sp]) amp = n ? __fdiv_rn(amp, (float)n) : 0.0f;
                    float2 *out = p.sig + (size_t)sp * p.M * p.D + (size_t)m * p.D;
                    if (dsel >= 0) out[dsel] = make_float2(amp, (float)kb);           // (tid < G: this thread's slot is d = tid)
                    // the mirrored histogram has the same amplitude spectrum
                    if (dpart >= 0 && !((s_mask >> tid) & 1u)) out[dpart] = make_float2(amp, (float)kb);
                }
                __syncthreads();                                          // cand is reused by the next spec
            }
            // the next group's clear of buf is ordered after this group's reads by the barrier above; cand is
            // rewritten only after three more barriers
            if (!fix) ++gi;
        }
      }
    }
}

static int fft_groups_of(int B) { return B <= 1024 ? 32 : 32768 / B; }
static size_t fft_smem_for(int B, int cap)
{
    const int G = fft_groups_of(B), T = kFftThreads / G;
    return (size_t)B * G * 4 + (size_t)(B / 2) * 8 + (size_t)T * G * 8 + (size_t)cap * 12;
}
static int fft_cap_for(int B)
{
    const size_t budget = 232448 - 1024;           // minus static shared (fix-up list, flags)
    return (int)(((budget - fft_smem_for(B, 0)) / 12) & ~(size_t)63);
}

// M = material points of the call (plane stride of the outputs); list != nullptr: only the listed ones are processed
static cudaError_t launch_fft_common(Plan *p, const float *centres, int64_t M, const uint32_t *list, float *sig,
                                     uint32_t *counts, cudaStream_t st)
{
    const int B = p->B, G = fft_groups_of(B);
    FftParams q;
    q.sorted = p->d_sorted; q.cell_start = p->d_cell_start; q.grid = p->d_grid; q.centres = centres;
    q.dirs_scaled = p->d_dirs_scaled; q.tw = p->d_twiddle; q.sig = reinterpret_cast<float2 *>(sig); q.counts = counts;
    q.hist_out = p->dbg_hist_out; q.hist_d0 = p->dbg_d0; q.hist_nd = p->dbg_nd;
    q.ss = p->specs; q.M = M;
    q.list = list; q.D = p->D; q.k_lo = p->k_lo; q.k_hi = p->k_hi; q.cap = fft_cap_for(B);
    // half-grid mode on antipodally symmetric grids (not under the histogram export hook, which indexes groups by direction)
    const bool halfmode = p->fft_paired && !p->dbg_hist_out;
    q.half = halfmode ? p->d_fft_half : nullptr; q.partner = halfmode ? p->d_fft_partner : nullptr; q.Dh = p->D / 2;
    q.ngroups = ((halfmode ? q.Dh : p->D) + G - 1) / G;
    // enough CTAs to fill the machine a few times over, but at least a handful of groups per CTA (one gather each)
    int nchunks = 1;
    const int64_t want = (int64_t)p->sm_count * 4;
    const int64_t Mx = list ? 1 : M;
    if (Mx * nchunks < want) nchunks = (int)((want + Mx - 1) / Mx);
    if (nchunks > (q.ngroups + 1) / 2) nchunks = (q.ngroups + 1) / 2;
    if (nchunks < 1) nchunks = 1;
    q.nchunks = nchunks;
    q.R = p->R; q.R2 = p->R2;
    q.clamp = p->need_clamp;
    const size_t smem = fft_smem_for(B, q.cap);
    const int64_t blocks = list ? (int64_t)p->sm_count : M * nchunks;
    if (blocks > 0x7FFFFFFFLL) return cudaErrorInvalidConfiguration;
    auto launch = [&](auto kern) -> cudaError_t {
        cudaError_t le = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (le != cudaSuccess) return le;
        kern<<<(unsigned)blocks, kFftThreads, smem, st>>>(q);
        return cudaGetLastError();
    };
    switch (B) {
        case 256: return halfmode ? launch(k_signature_fft<256, true>) : launch(k_signature_fft<256, false>);
        case 512: return halfmode ? launch(k_signature_fft<512, true>) : launch(k_signature_fft<512, false>);
        case 1024: return halfmode ? launch(k_signature_fft<1024, true>) : launch(k_signature_fft<1024, false>);
        case 2048: return halfmode ? launch(k_signature_fft<2048, true>) : launch(k_signature_fft<2048, false>);
        case 4096: return halfmode ? launch(k_signature_fft<4096, true>) : launch(k_signature_fft<4096, false>);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_signature_fft(Plan *p, const float *centres, int64_t M, float *sig, uint32_t *counts,
                                 cudaStream_t st)
{
    if (M == 0) return cudaSuccess;
    return launch_fft_common(p, centres, M, nullptr, sig, counts, st);
}

cudaError_t launch_signature_fft_list(Plan *p, const float *centres, const uint32_t *list, int64_t M, float *sig,
                                      uint32_t *counts, cudaStream_t st)
{
    return launch_fft_common(p, centres, M, list, sig, counts, st);
}

}  // namespace apx
