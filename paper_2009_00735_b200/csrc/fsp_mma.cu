// fsp_mma.cu -- reciprocal space method (Eq. 2) on the tensor cores (tcgen05 + TMEM).
//
// One z-slice pair of the image of one material point is the complex contraction (fsp.cu)
//     C[(iz, iy)][ix] = sum_w (ez_w[iz] ey_w[iy]) * ex_w[ix]            (phases factorise per axis),
// written as ONE real GEMM with the complex parts stacked:  rows m = (iz_local, iy) (2 x 64 = 128), K index k' = (w, part)
// (part = re / im of the A factor), columns n' = (part', ix) (2 x 64 = 128):
//     A'[m][(w,re)] = Re a,  A'[m][(w,im)] = Im a,            a = ez_w ey_w
//     B'[(w,re)][(re,ix)] = Re e,  B'[(w,im)][(re,ix)] = -Im e,  B'[(w,re)][(im,ix)] = Im e,  B'[(w,im)][(im,ix)] = Re e,   e = ex_w[ix]
// so that C'[m][(re,ix)] = Re C and C'[m][(im,ix)] = Im C.  Operands are fp16; to keep fp32-level accuracy every operand is
// split x = hi + 2^-11 lo (both fp16) and three products are accumulated in fp32 in TMEM:
//     D0 += Ah Bh,   D1 += Ah Bl + Al Bh,   C' = D0 + D1 / 2048        (the lo*lo term, 2^-22 relative, is dropped).
// CTA = (material point, TWO pairs of z-slices, 64 x 64 tile of (iy, ix)): the B' tiles and the ey / ex factors of a chunk are
// built once and feed both pairs (each pair has its own A tiles and its own D0 / D1 accumulators: 4 x 128 = all 512 TMEM
// columns); ions in chunks of 32 (K' = 64 = one 128-byte swizzle row).  All 512 threads build the four operand tiles of a chunk (phase factors by sincospif, exact argument reduction) in
// one of two shared-memory stages, one thread issues the 24 tcgen05.mma of the chunk and commits to the stage's mbarrier;
// building chunk c+1 overlaps the MMAs of chunk c.  ROIs with more ions than the shared buffer are left to k_fsp (fsp.cu).
#include <cuda_fp16.h>
#include "common.cuh"
#include "../../include/aptsig_ext.h"

namespace apx {

constexpr int kFmThreads = 512;                // threads that build the operand tiles (16 warps)
constexpr int kFmAll = kFmThreads + 32;         // + one warp that only issues the MMAs, so that no builder arrives late at the
                                                // chunk barrier because it had the tensor-core instructions to issue
constexpr int kFmPer = 64 / (kFmThreads / 32);   // consecutive iy / ix per thread when the operand tiles are built
constexpr int kFmChunk = 32;                  // ions per chunk
constexpr int kFmTileBytes = 128 * 128;       // 128 rows x 64 fp16 (K-major, SWIZZLE_128B)
constexpr int kFmPairs = 2;                   // z-slice pairs per CTA: one B' tile and one set of ey / ex factors feed all of them
constexpr int kFmSlices = 2 * kFmPairs;
constexpr int kFmStageBytes = (2 * kFmPairs + 2) * kFmTileBytes;   // (Ah, Al) per slice pair, Bh, Bl
constexpr int kFmCap = 2560;                  // ions held in shared memory beside the two stages

struct FspMmaParams {
    const float4 *sorted;
    const uint32_t *cell_start;
    const GridParams *grid;
    const float *centres;
    const float *kaxis;
    float dk;                 // spacing of the k axis
    float *out;
    uint32_t *counts;
    uint32_t *list;           // [0] = count, [1..] = material points left to k_fsp (more than `cap` ions)
    int L, tiles, cap;
    float R, R2;
};

__device__ __forceinline__ uint32_t fm_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fm_mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done, spins = 0;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(fm_smem_u32(bar)), "r"(parity), "r"(1000000u) : "memory");
        if (!done && ++spins > (1u << 22)) asm volatile("trap;");          // never hang the device on a lost commit
    } while (!done);
}
__device__ __forceinline__ void fm_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc)
{
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void fm_tmem_ld16(uint32_t addr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(addr));
}
// x = hi + lo / 2048 with hi, lo fp16; packed as (hi, lo) in the low / high halves of the result
__device__ __forceinline__ void fm_split(float x, uint16_t &hi, uint16_t &lo)
{
    const __half h = __float2half_rn(x);
    const __half l = __float2half_rn((x - __half2float(h)) * 2048.0f);
    hi = __half_as_ushort(h); lo = __half_as_ushort(l);
}
// two values at once: (a, b) -> hi = half2(a, b), lo = half2((a - hi.a) * 2048, (b - hi.b) * 2048), a in the low half
__device__ __forceinline__ void fm_split2(float a, float b, uint32_t &hi, uint32_t &lo)
{
    // lo = rn16((a - hi) * 2048): a - hi is exact in fp32 and so is the scaling, hence fma(a, 2048, -2048 * hi) -- with
    // -2048 * hi formed exactly on the packed halves -- is the same number in one rounding-free step less per value
    const __half2 h = __floats2half2_rn(a, b);
    const float2 hs = __half22float2(__hmul2(h, __floats2half2_rn(-2048.0f, -2048.0f)));
    const __half2 l = __floats2half2_rn(__fmaf_rn(a, 2048.0f, hs.x), __fmaf_rn(b, 2048.0f, hs.y));
    hi = *reinterpret_cast<const uint32_t *>(&h);
    lo = *reinterpret_cast<const uint32_t *>(&l);
}
// byte offset of (row r, K pair index j = ion within the chunk) in a K-major SWIZZLE_128B tile: 128-byte rows, the 16-byte
// chunk index (j / 4) XORed with (r & 7); a pair (re, im) of fp16 is one 32-bit word
__device__ __forceinline__ uint32_t fm_off(int r, int j) { return (uint32_t)r * 128u + (uint32_t)((((j >> 2) ^ (r & 7)) << 4) + ((j & 3) << 2)); }

__device__ __forceinline__ float2 fm_phase(float k, float d)
{
    float s, c;
    sincospif(-2.0f * __fmul_rn(k, d), &s, &c);
    return make_float2(c, s);
}

// Operand tiles of one chunk (see the kernel).  off[u] = byte offset of (row kFmPer * seg + u, K pair j) in a tile, computed
// once per CTA: the rows 64 further down (second z-slice of A, imaginary block of B) sit exactly 8192 bytes behind, because
// the swizzle only looks at the row index modulo 8.
template <bool kFull>
__device__ __forceinline__ void fm_build_tiles(const FspMmaParams &p, unsigned char *A, unsigned char *Bh,
                                               unsigned char *Bl, const float *ions, const float2 (*s_ion)[kFmChunk],
                                               const uint32_t (&off)[kFmPer], int w0, int n, int iy0, int ix0, int L, int tid)
{
    const int j = tid & 31, seg = tid >> 5;
    const bool ion_ok = kFull || w0 + j < n;
    const float dx = ion_ok ? ions[3 * (w0 + j)] : 0.f, dy = ion_ok ? ions[3 * (w0 + j) + 1] : 0.f;
    float2 ez[kFmSlices];
#pragma unroll
    for (int zl = 0; zl < kFmSlices; ++zl) ez[zl] = s_ion[zl][j];                 // (zero for a missing ion / slice)
    const float2 ry = s_ion[kFmSlices][j], rx = s_ion[kFmSlices + 1][j];
    float2 ey = fm_phase(p.kaxis[min(iy0 + kFmPer * seg, L - 1)], dy), ex = fm_phase(p.kaxis[min(ix0 + kFmPer * seg, L - 1)], dx);
#pragma unroll
    for (int u = 0; u < kFmPer; ++u) {
        const int t64 = kFmPer * seg + u;
        const bool y_ok = kFull || (ion_ok && iy0 + t64 < L), x_ok = kFull || (ion_ok && ix0 + t64 < L);
#pragma unroll
        for (int zl = 0; zl < kFmSlices; ++zl) {
            const float ar = y_ok ? ez[zl].x * ey.x - ez[zl].y * ey.y : 0.f, ai = y_ok ? ez[zl].x * ey.y + ez[zl].y * ey.x : 0.f;
            uint32_t hi, lo;
            fm_split2(ar, ai, hi, lo);
            unsigned char *Ah = A + (zl >> 1) * (2 * kFmTileBytes), *Al = Ah + kFmTileBytes;      // tiles of slice pair zl / 2
            *reinterpret_cast<uint32_t *>(Ah + off[u] + (zl & 1) * 8192u) = hi;
            *reinterpret_cast<uint32_t *>(Al + off[u] + (zl & 1) * 8192u) = lo;
        }
        {
            uint32_t hi, lo;                                       // (Re e, Im e) in (low, high) halves
            fm_split2(x_ok ? ex.x : 0.f, x_ok ? ex.y : 0.f, hi, lo);
            *reinterpret_cast<uint32_t *>(Bh + off[u]) = hi ^ 0x80000000u;                    // (Re e, -Im e)
            *reinterpret_cast<uint32_t *>(Bl + off[u]) = lo ^ 0x80000000u;
            *reinterpret_cast<uint32_t *>(Bh + off[u] + 8192u) = __byte_perm(hi, 0, 0x1032);    // (Im e,  Re e)
            *reinterpret_cast<uint32_t *>(Bl + off[u] + 8192u) = __byte_perm(lo, 0, 0x1032);
        }
        const float2 ny = make_float2(ey.x * ry.x - ey.y * ry.y, ey.x * ry.y + ey.y * ry.x);
        const float2 nx = make_float2(ex.x * rx.x - ex.y * rx.y, ex.x * rx.y + ex.y * rx.x);
        ey = ny; ex = nx;
    }
}

__global__ void __launch_bounds__(kFmAll, 1) k_fsp_mma(const __grid_constant__ FspMmaParams p)
{
    extern __shared__ unsigned char fm_raw[];
    unsigned char *smem = fm_raw + ((1024u - (fm_smem_u32(fm_raw) & 1023u)) & 1023u);      // 1024-byte aligned (swizzle atoms)
    unsigned char *stage0 = smem;                                         // [2][Ah | Al | Bh | Bl]
    float *ions = reinterpret_cast<float *>(smem + 2 * kFmStageBytes);    // [cap][3]
    __shared__ uint64_t s_done[2], s_final;
    __shared__ uint32_t s_tmem;
    __shared__ int s_n;
    __shared__ float2 s_ion[2][kFmSlices + 2][kFmChunk];   // per ion of a chunk: ez of the CTA's slices, step factors along y, x;
                                                            // [c & 1]: chunk c's are computed while chunk c - 1 is built

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int L = p.L;
    int b = blockIdx.x;
    const int tx_tile = b % p.tiles; b /= p.tiles;
    const int ty_tile = b % p.tiles; b /= p.tiles;
    const int nzp = (L + kFmSlices - 1) / kFmSlices;         // groups of kFmSlices z-slices
    const int izp = b % nzp;
    const int64_t m = b / nzp;
    const int iz0 = kFmSlices * izp, iy0 = ty_tile * 64, ix0 = tx_tile * 64;
    const GridParams g = *p.grid;
    const float cx = p.centres[3 * m], cy = p.centres[3 * m + 1], cz = p.centres[3 * m + 2];
    const RoiCells rc = roi_cells(g, cx, cy, cz, p.R);

    if (tid == 0) {
        for (int i = 0; i < 2; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(fm_smem_u32(&s_done[i])));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(fm_smem_u32(&s_final)));
        asm volatile("fence.mbarrier_init.release.cluster;");
        s_n = 0;
    }
    if (wid == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(fm_smem_u32(&s_tmem)), "r"(256u * kFmPairs));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = s_tmem;

    // ---- gather (as in fsp.cu) ------------------------------------------------------------------------------------
    const bool builder = wid < kFmThreads / 32;
    if (g.n_accepted && builder) {
        const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
        for (int row = wid; row < ny_r * nz_r; row += kFmThreads / 32) {
            const int iy = rc.iy0 + row % ny_r, izc = rc.iz0 + row / ny_r;
            const int base = (izc * g.ny + iy) * g.nx;
            const uint32_t beg = p.cell_start[base + rc.ix0], end = p.cell_start[base + rc.ix1 + 1];
            for (uint32_t i = beg + lane; i < ((end - beg + 31u) & ~31u) + beg; i += 32) {
                bool in = false;
                float dx = 0.f, dy = 0.f, dz = 0.f;
                if (i < end) {
                    const float4 q = p.sorted[i];
                    dx = __fsub_rn(q.x, cx); dy = __fsub_rn(q.y, cy); dz = __fsub_rn(q.z, cz);
                    in = inside(dx, dy, dz, p.R2);
                }
                const unsigned msk = __ballot_sync(0xffffffffu, in);
                if (msk) {
                    int pos = 0;
                    if (lane == 0) pos = atomicAdd(&s_n, __popc(msk));
                    pos = __shfl_sync(0xffffffffu, pos, 0) + __popc(msk & ((1u << lane) - 1u));
                    if (in && pos < p.cap) { ions[3 * pos] = dx; ions[3 * pos + 1] = dy; ions[3 * pos + 2] = dz; }
                }
            }
        }
    }
    __syncthreads();
    const int n = s_n;
    if (p.counts && izp == 0 && tx_tile == 0 && ty_tile == 0 && tid == 0) p.counts[m] = (uint32_t)n;
    const bool skip = n > p.cap;                           // too many ions for the shared buffer: k_fsp serves this ROI
    if (skip && izp == 0 && tx_tile == 0 && ty_tile == 0 && tid == 0) p.list[1 + atomicAdd(&p.list[0], 1u)] = (uint32_t)m;

    // instruction descriptor: D = f32, A = B = f16, both K-major, N = 128, M = 128
    const uint32_t idesc = (1u << 4) | ((uint32_t)(128 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    const uint32_t d_hi = (uint32_t)(1024 >> 4) | (1u << 14) | (2u << 29);                  // SBO = 1024 B, version 1, SWIZZLE_128B
    const int nchunks = skip ? 0 : (n + kFmChunk - 1) / kFmChunk;
    const bool z_all_valid = iz0 + kFmSlices <= L;

    uint32_t tile_off[kFmPer];
#pragma unroll
    for (int u = 0; u < kFmPer; ++u) tile_off[u] = fm_off(kFmPer * (tid >> 5) + u, tid & 31);
    // per-ion factors of chunk c, computed once: phases along z for the CTA's slices and the step factors exp(-2 pi i dk d)
    // along y and x (sincospif: exact argument reduction).  One factor per thread (the first 192 threads); chunk c + 1's are
    // computed behind the tile build of chunk c and published by its barrier.
    auto ion_factors = [&](int c) {
        if (tid < (kFmSlices + 2) * kFmChunk) {
            const int j = tid & (kFmChunk - 1), which = tid / kFmChunk, w0 = c * kFmChunk;
            float2 e = make_float2(0.f, 0.f);
            if (w0 + j < n) {
                if (which < kFmSlices) e = iz0 + which < L ? fm_phase(p.kaxis[min(iz0 + which, L - 1)], ions[3 * (w0 + j) + 2]) : e;
                else if (which == kFmSlices) e = fm_phase(p.dk, ions[3 * (w0 + j) + 1]);
                else e = fm_phase(p.dk, ions[3 * (w0 + j)]);
            }
            s_ion[c & 1][which][j] = e;
        }
    };
    for (int c = 0; c < nchunks; ++c) {
        const int s = c & 1, use = c >> 1;
        if (builder && use >= 1) fm_mbar_wait(&s_done[s], (uint32_t)((use - 1) & 1));   // the MMAs that read this stage have completed
        unsigned char *A = stage0 + s * kFmStageBytes, *Bh = A + 2 * kFmPairs * kFmTileBytes, *Bl = Bh + kFmTileBytes;
        const int w0 = c * kFmChunk;
        if (c == 0) {
            if (builder) ion_factors(0);
            __syncthreads();
        }
        // thread = (ion j of the chunk, kFmPer consecutive iy and ix): the phase factor of the first one comes from sincospif,
        // the next ones by multiplying with the step factor -- a few fp32 complex products add < 4e-7 to the phase, inside the
        // tolerance budget of DESIGN.md section 2.  A warp writes one 128-byte operand row per store (32 consecutive K pairs):
        // conflict-free.  Splits x = hi + lo / 2048 are taken two values at a time (cvt.rn.f16x2.f32).  A chunk of 32 ions in a
        // tile that lies inside the k grid (the common case) takes the copy without the validity selects.
        if (builder) {
            const bool full = w0 + kFmChunk <= n && iy0 + 64 <= L && ix0 + 64 <= L && z_all_valid;
            if (full) fm_build_tiles<true>(p, A, Bh, Bl, ions, s_ion[c & 1], tile_off, w0, n, iy0, ix0, L, tid);
            else fm_build_tiles<false>(p, A, Bh, Bl, ions, s_ion[c & 1], tile_off, w0, n, iy0, ix0, L, tid);
            if (c + 1 < nchunks) ion_factors(c + 1);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");       // operand tiles -> async proxy (tensor core)
        asm volatile("tcgen05.fence::before_thread_sync;");
        __syncthreads();
        if (tid == kFmThreads) {                                           // (first lane of the issuing warp)
            asm volatile("tcgen05.fence::after_thread_sync;");
            const uint32_t bh = (fm_smem_u32(Bh) >> 4) & 0x3FFFu, bl = (fm_smem_u32(Bl) >> 4) & 0x3FFFu;
#pragma unroll
            for (int pr = 0; pr < kFmPairs; ++pr) {             // slice pair pr: its own A tiles and accumulators, the shared B' tiles
                const uint32_t ah = (fm_smem_u32(A + pr * 2 * kFmTileBytes) >> 4) & 0x3FFFu, al = ah + (uint32_t)(kFmTileBytes >> 4);
                const uint32_t acc = tmem + 256u * (uint32_t)pr;
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {                // K = 16 per MMA: +32 bytes inside the 128-byte swizzle row
                    const uint32_t adv = (uint32_t)ks * 2u;
                    const uint64_t dAh = ((uint64_t)d_hi << 32) | ((ah + adv) | (1u << 16)), dAl = ((uint64_t)d_hi << 32) | ((al + adv) | (1u << 16));
                    const uint64_t dBh = ((uint64_t)d_hi << 32) | ((bh + adv) | (1u << 16)), dBl = ((uint64_t)d_hi << 32) | ((bl + adv) | (1u << 16));
                    const uint32_t first = (c == 0 && ks == 0) ? 0u : 1u;
                    fm_mma(acc, dAh, dBh, idesc, first);            // D0 += Ah Bh
                    fm_mma(acc + 128u, dAh, dBl, idesc, first);     // D1 += Ah Bl
                    fm_mma(acc + 128u, dAl, dBh, idesc, 1u);        // D1 += Al Bh
                }
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(fm_smem_u32(&s_done[s])) : "memory");
            if (c == nchunks - 1)
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(fm_smem_u32(&s_final)) : "memory");
        }
    }

    // ---- epilogue: |C'| -> out[m][iz][iy][ix]; warps 0..3 own TMEM lane quarters = rows (iz_local = q / 2, iy = 32 (q & 1) + lane)
    //      of every slice pair; pair pr has its accumulators at columns 256 pr
    if (!skip && wid < 4) {
        if (nchunks > 0) {
            fm_mbar_wait(&s_final, 0u);
            asm volatile("tcgen05.fence::after_thread_sync;");
        }
#pragma unroll 1
        for (int pr = 0; pr < kFmPairs; ++pr) {
            const int zl = 2 * pr + (wid >> 1), iy = iy0 + 32 * (wid & 1) + lane, iz = iz0 + zl;
            const bool row_ok = iz < L && iy < L;
            float *o = p.out + (((size_t)m * L + min(iz, L - 1)) * L + min(iy, L - 1)) * (size_t)L + ix0;
            if (nchunks > 0) {
                const uint32_t row_addr = tmem + 256u * (uint32_t)pr + ((uint32_t)(wid * 32) << 16);
#pragma unroll 1
                for (int cb = 0; cb < 4; ++cb) {                  // 16 ix per step: Re at columns ix, Im at 64 + ix, D1 at +128
                    uint32_t r0[16], r1[16], i0[16], i1[16];
                    fm_tmem_ld16(row_addr + (uint32_t)(16 * cb), r0);
                    fm_tmem_ld16(row_addr + (uint32_t)(128 + 16 * cb), r1);
                    fm_tmem_ld16(row_addr + (uint32_t)(64 + 16 * cb), i0);
                    fm_tmem_ld16(row_addr + (uint32_t)(192 + 16 * cb), i1);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        const float re = __uint_as_float(r0[e]) + __uint_as_float(r1[e]) * (1.0f / 2048.0f);
                        const float im = __uint_as_float(i0[e]) + __uint_as_float(i1[e]) * (1.0f / 2048.0f);
                        const int ix = ix0 + 16 * cb + e;
                        if (row_ok && ix < L) o[16 * cb + e] = sqrtf(re * re + im * im);
                    }
                }
            } else if (row_ok) {                                 // empty ROI: F = 0
                for (int e = 0; e < 64; ++e)
                    if (ix0 + e < L) o[e] = 0.f;
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (wid == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(256u * kFmPairs));
}

// launcher (called by apx_fsp)
cudaError_t launch_fsp_mma(Plan *p, const float *centres, int64_t M, int L, float dk, float *out, uint32_t *counts, uint32_t *list,
                           cudaStream_t st)
{
    FspMmaParams q;
    q.sorted = p->d_sorted; q.cell_start = p->d_cell_start; q.grid = p->d_grid; q.centres = centres; q.kaxis = p->d_kaxis;
    q.out = out; q.counts = counts; q.list = list; q.L = L; q.tiles = (L + 63) / 64; q.cap = kFmCap; q.R = p->R; q.R2 = p->R2; q.dk = dk;
    const int64_t blocks = M * ((L + kFmSlices - 1) / kFmSlices) * q.tiles * q.tiles;
    if (blocks > 0x7FFFFFFFLL) return cudaErrorInvalidConfiguration;
    const size_t smem = 2 * (size_t)kFmStageBytes + (size_t)q.cap * 12 + 1024;
    cudaError_t e = cudaFuncSetAttribute(k_fsp_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_fsp_mma<<<(unsigned)blocks, kFmAll, smem, st>>>(q);
    return cudaGetLastError();
}

// The same launch with the k axis at a caller-given device address instead of the plan's d_kaxis: used by apx_fsp_noalloc
// (fsp.cu), whose k axis and deferred list live in the library's static scratch array.
cudaError_t launch_fsp_mma_at(Plan *p, const float *kaxis, const float *centres, int64_t M, int L, float dk, float *out,
                              uint32_t *counts, uint32_t *list, cudaStream_t st)
{
    FspMmaParams q;
    q.sorted = p->d_sorted; q.cell_start = p->d_cell_start; q.grid = p->d_grid; q.centres = centres; q.kaxis = kaxis;
    q.out = out; q.counts = counts; q.list = list; q.L = L; q.tiles = (L + 63) / 64; q.cap = kFmCap; q.R = p->R; q.R2 = p->R2; q.dk = dk;
    const int64_t blocks = M * ((L + kFmSlices - 1) / kFmSlices) * q.tiles * q.tiles;
    if (blocks > 0x7FFFFFFFLL) return cudaErrorInvalidConfiguration;
    const size_t smem = 2 * (size_t)kFmStageBytes + (size_t)q.cap * 12 + 1024;
    cudaError_t e = cudaFuncSetAttribute(k_fsp_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_fsp_mma<<<(unsigned)blocks, kFmAll, smem, st>>>(q);
    return cudaGetLastError();
}

}  // namespace apx
