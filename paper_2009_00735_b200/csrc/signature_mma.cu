// signature_mma.cu -- windowed-DFT signature kernel: shared-memory histograms feed the tcgen05 tensor
// cores directly (steps a2, a4-a7 for narrow spectral windows, B <= 1024).
//
// Per CTA: one material point x a chunk of direction groups; a group = 64 directions.
//   binning  : every lane of a binning warp owns ONE 32-bit word per histogram row: two u16 counters, the
//              low half for direction `lane` (set A) and the high half for direction `lane + 32` (set B) of
//              the group (Eq. 1).  A row of the histogram is 32 words, so within one shared
//              atomic the 32 lanes hit 32 different banks whenever their bins agree in the top three bits
//              (hi3); the plan sorts the directions into spatially compact patches of 32 so that they
//              almost always do.  The u16 bit pattern c is the fp16 number c * 2^-24 (subnormal / first
//              binade, exact for c <= 2048), so the histogram IS a valid fp16 tensor-core operand and is
//              never converted or copied.
//   layout   : byte address of (bin b, lane L) = (L/4)*144 + (L%4)*4 + 16*hi3 + 1152*low,
//              hi3 = b >> (log2 B - 3), low = b & (B/8 - 1).  Read as an MN-major INTERLEAVE (no swizzle)
//              operand with SBO = 144 B (between 8-element M chunks) and LBO = 2304 B (between 8-row K
//              groups) this is a [128 x K] tile: M row = blk*64 + direction slot (blk = bit 0 of low),
//              K index = kg*8 + hi3 (kg = the middle bits of low); the top bit of low selects one of two
//              accumulators ("pair").  K = B/4 per accumulator.
//   DFT      : X_k = sum_b h_b w^{bk} restricted to the window [k_lo,k_hi] is the dense contraction
//              [directions x bins] x [bins x window] (L73, L75).  With b = hi3*B/8 + 2*kg + (pair*B/16 + blk)
//              the four (pair, blk) parts share one twiddle table T[k=(kg,hi3)][n] and are recombined in the
//              epilogue with the phases w^{(pair*B/16+blk) k}.  T holds cos/sin as fp16 hi + lo parts
//              (columns 4w+{0,1,2,3} = cos_hi, sin_hi, 2^11 cos_lo, 2^11 sin_lo) so amplitudes reach ~1e-7.
//   peak     : |X_k|^2 arg-max over the window, lowest k on ties (L75, L416); A* = 2^24 sqrt(max).
// One histogram buffer (144*B bytes): bin -> transform -> clear are serial per group; the epilogue of
// group g runs while group g+1 is binned.  ROIs with more ions than the shared-memory ion buffer are
// appended to a deferred list and handled by the general FFT kernel.
#include <algorithm>
#include <cmath>
#include <cuda_fp16.h>
#include <numeric>
#include <vector>
#include "common.cuh"

namespace apx {

constexpr int kEpiWarps = 4;             // warps 0..3 = epilogue (one per TMEM lane quarter)
constexpr int kMmaWarp = 4;              // tcgen05.mma issuer
constexpr int kFirstBinWarp = 5;
constexpr int kBinWarps = 12;            // project-and-bin warps (3 per scheduler)
constexpr int kMmaWarps = kFirstBinWarp + kBinWarps;
constexpr int kMmaThreads = kMmaWarps * 32;
constexpr int kBinThreads = kBinWarps * 32;
constexpr int kIonBatch = 8;
constexpr int kRowGroupBytes = 1152;     // 8 M-chunks of 144 B: one (blk, kg) slab of 8 K rows x 64 directions
constexpr int kChunkBytes = 144;         // SBO: 8 directions x 8 rows x 2 B + 16 B skew

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t cnt)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(cnt));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    uint32_t spins = 0;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (!done && ++spins > (1u << 24)) asm volatile("trap;");     // never hang the device on a lost commit
    } while (!done);
}
// shared-memory matrix descriptor (tcgen05): start address, leading / stride byte offsets (16-byte units),
// descriptor version 1, layout type in bits 61-63 (0 = INTERLEAVE / no swizzle, 2 = 128B, 4 = 64B)
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout)
{
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46) | ((uint64_t)layout << 61);
}
__device__ __forceinline__ void mma_f16_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc)
{
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void red_shared_add(uint32_t addr, uint32_t v)
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ float4 lds128(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void tmem_ld16(uint32_t addr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(addr));
}

struct MmaParams {
    const float4 *sorted;
    const uint32_t *cell_start;
    const GridParams *grid;
    const float *centres;
    const float *dirs_sorted;  // [Dp][3] scaled directions in patch order (Dp = D rounded up to 64)
    const int *perm;           // [Dp] original direction index of each sorted slot, -1 = padding
    const uint4 *table;        // pre-swizzled twiddle operand image, (K/64) blocks of [N][128 B]
    const float2 *phase;       // [4][W] recombination phases, index pair*2 + blk
    float2 *sig;
    uint32_t *counts;
    uint32_t *deferred;        // [0] = count, [1..] = material point ids left to the FFT kernel
    int D, B, nl, k_lo, W, N, cap, nchunks, ngroups, clamp;
    uint32_t tmem_cols;
    float R, R2;
};

// smem carve-up (bytes), shared by host and device
struct MmaSmem {
    uint32_t table, hist, exch, phase, ions, total;
};
__host__ __device__ inline MmaSmem mma_smem_layout(int B, int N, int W, int cap)
{
    MmaSmem s;
    uint32_t off = 0;
    s.table = off; off += (uint32_t)(B / 4) * N * 2;             // (K/64) * N * 128 with K = B/4; multiple of 1024
    s.hist = off; off += (uint32_t)B * kChunkBytes;              // (B/8) row groups of 1152 B
    s.exch = off; off += 64u * W * 8;
    s.phase = off; off += 4u * W * 8;
    s.ions = off; off += (uint32_t)cap * 16;
    s.total = off + 1024;                                          // slack for 1024-byte alignment
    return s;
}

// Gather (step a2) into float4 records (dx, dy, dz, -) for warp-broadcast LDS.128 reads.
__device__ __forceinline__ void gather_roi4(const MmaParams &p, const GridParams &g, const RoiCells &rc,
                                            float cx, float cy, float cz, float4 *ions, int *s_n)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
    for (int row = wid; row < ny_r * nz_r; row += kMmaWarps) {
        int iy = rc.iy0 + row % ny_r, iz = rc.iz0 + row / ny_r;
        int base = (iz * g.ny + iy) * g.nx;
        uint32_t beg = p.cell_start[base + rc.ix0], end = p.cell_start[base + rc.ix1 + 1];
        for (uint32_t i = beg + lane; i < ((end - beg + 31u) & ~31u) + beg; i += 32) {
            bool in = false;
            float dx = 0.f, dy = 0.f, dz = 0.f;
            if (i < end) {
                float4 q = p.sorted[i];
                dx = __fsub_rn(q.x, cx); dy = __fsub_rn(q.y, cy); dz = __fsub_rn(q.z, cz);
                in = inside(dx, dy, dz, p.R2);
            }
            unsigned msk = __ballot_sync(0xffffffffu, in);
            if (msk) {
                int pos = 0;
                if (lane == 0) pos = atomicAdd(s_n, __popc(msk));
                pos = __shfl_sync(0xffffffffu, pos, 0) + __popc(msk & ((1u << lane) - 1u));
                if (in && pos < p.cap) ions[pos] = make_float4(dx, dy, dz, 0.f);
            }
        }
    }
}

// Project-and-bin (step a4) of one ion for one direction of this lane.
//   ua = bits(RD(x + 1.5*2^23 + B/2))       = 0x4B400000 + b          (b = B/2 + floor(x), Eq. 1)
//   va = bits(RD(x*2^-nl + 1.5*2^23 + 4))   = 0x4B400000 + hi3        (hi3 = b >> nl, exact: floor(floor(y)/n) = floor(y/n))
//   address = hist + lane offset + 1152*low + 16*hi3 = ua*1152 + va*(16 - 1152*2^nl) + k0   (mod 2^32)
struct BinConst {
    float half_b, magic_a, magic_b, scl;
    uint32_t kz, k0;
};
template <bool kClamp>
__device__ __forceinline__ void bin_one(const float4 q, float npx, float npy, float npz, const BinConst &c, uint32_t inc)
{
    float x = __fmaf_rn(npz, q.z, __fmaf_rn(npy, q.y, __fmul_rn(npx, q.x)));
    if (kClamp) x = fminf(fmaxf(x, -c.half_b), c.half_b - 0.25f);
    const uint32_t ua = __float_as_uint(__fadd_rd(x, c.magic_a));
    const uint32_t va = __float_as_uint(__fmaf_rd(x, c.scl, c.magic_b));
    red_shared_add(ua * (uint32_t)kRowGroupBytes + (va * c.kz + c.k0), inc);
}

// ions_s = shared-space byte address of the float4 ion records; A = direction `lane`, B = direction `lane+32`
template <bool kClamp>
__device__ __forceinline__ void bin_ions(uint32_t ions_s, int i0, int i1, const float (&na)[3], const float (&nb)[3],
                                         const BinConst &c)
{
    int ib = i0;
    for (; ib + kIonBatch <= i1; ib += kIonBatch) {          // full batches: loads first, then 16 independent chains
        float4 q[kIonBatch];
#pragma unroll
        for (int u = 0; u < kIonBatch; ++u) q[u] = lds128(ions_s + (uint32_t)(ib + u) * 16u);
#pragma unroll
        for (int u = 0; u < kIonBatch; ++u) {
            bin_one<kClamp>(q[u], na[0], na[1], na[2], c, 1u);
            bin_one<kClamp>(q[u], nb[0], nb[1], nb[2], c, 65536u);
        }
    }
    for (; ib < i1; ++ib) {
        const float4 q = lds128(ions_s + (uint32_t)ib * 16u);
        bin_one<kClamp>(q, na[0], na[1], na[2], c, 1u);
        bin_one<kClamp>(q, nb[0], nb[1], nb[2], c, 65536u);
    }
}

__global__ void __launch_bounds__(kMmaThreads, 1) k_signature_mma(const MmaParams p)
{
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 1024-byte aligned, still shared-space
    const MmaSmem L = mma_smem_layout(p.B, p.N, p.W, p.cap);
    __shared__ uint64_t s_full, s_done, s_tfree;
    __shared__ uint32_t s_tmem;
    __shared__ int s_n;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t m = blockIdx.x / p.nchunks;
    const int chunk = blockIdx.x % p.nchunks;
    const int g_begin = (int)((int64_t)chunk * p.ngroups / p.nchunks);
    const int g_end = (int)((int64_t)(chunk + 1) * p.ngroups / p.nchunks);
    const GridParams g = *p.grid;
    const float cx = p.centres[3 * m], cy = p.centres[3 * m + 1], cz = p.centres[3 * m + 2];
    const RoiCells rc = roi_cells(g, cx, cy, cz, p.R);
    float4 *ions = reinterpret_cast<float4 *>(smem + L.ions);
    float2 *exch = reinterpret_cast<float2 *>(smem + L.exch);
    float2 *phase = reinterpret_cast<float2 *>(smem + L.phase);
    const int K = p.B / 4;
    const uint32_t hist_bytes = (uint32_t)p.B * kChunkBytes;

    // ---- setup: barriers, TMEM, zero histogram, twiddle table, gather ------------------------------
    if (tid == 0) {
        mbar_init(&s_full, kBinWarps);
        mbar_init(&s_done, 1);
        mbar_init(&s_tfree, kEpiWarps);
        asm volatile("fence.mbarrier_init.release.cluster;");
        s_n = 0;
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(p.tmem_cols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    {
        uint4 *h = reinterpret_cast<uint4 *>(smem + L.hist);
        for (int i = tid; i < (int)(hist_bytes / 16); i += kMmaThreads) h[i] = make_uint4(0, 0, 0, 0);
        uint4 *t = reinterpret_cast<uint4 *>(smem + L.table);
        for (int i = tid; i < K * p.N / 8; i += kMmaThreads) t[i] = p.table[i];
        for (int i = tid; i < 4 * p.W; i += kMmaThreads) phase[i] = p.phase[i];
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = s_tmem;
    if (g.n_accepted) gather_roi4(p, g, rc, cx, cy, cz, ions, &s_n);
    __syncthreads();
    const int n = s_n;
    if (chunk == 0 && tid == 0 && p.counts) p.counts[m] = (uint32_t)n;

    if (n > p.cap) {
        // too many ions for the shared buffer: leave this material point to the FFT kernel
        if (chunk == 0 && tid == 0) p.deferred[1 + atomicAdd(&p.deferred[0], 1u)] = (uint32_t)m;
    } else {
        // Warp-specialised pipeline over items = (direction group, ion pass), one histogram buffer:
        //   binning warps : wait done[it-1] -> clear the histogram -> project-and-bin item it -> arrive full
        //   MMA warp      : wait full, tfree[it-1] -> 2 x K/16 tcgen05.mma into the two accumulators -> commit to done
        //   epilogue warps: wait done[it]; on the last pass read TMEM, recombine the four (pair, blk) parts,
        //                    arg-max, store; arrive tfree
        const int npass = n > 2048 ? (n + 2047) / 2048 : 1;          // fp16 counters are exact up to 2048
        const int nitems = (g_end - g_begin) * npass;
        if (warp >= kFirstBinWarp) {
            const int bw = warp - kFirstBinWarp, bt = tid - kFirstBinWarp * 32;
            BinConst c;
            c.half_b = (float)(p.B / 2); c.magic_a = magic_for(p.B); c.magic_b = 12582912.0f + 4.0f;
            c.scl = __int_as_float((127 - p.nl) << 23);                       // 2^-nl
            c.kz = 16u - (uint32_t)kRowGroupBytes * (1u << p.nl);
            c.k0 = smem_u32(smem + L.hist) + (uint32_t)(lane >> 2) * kChunkBytes + (uint32_t)(lane & 3) * 4u
                   - 0x4B400000u * (uint32_t)kRowGroupBytes - 0x4B400000u * c.kz;
            const uint32_t ions_s = smem_u32(ions);
            for (int it = 0; it < nitems; ++it) {
                const int gi = g_begin + it / npass, pass = it % npass;
                float na[3], nb[3];
                {
                    const float *da = p.dirs_sorted + (size_t)(gi * 64 + lane) * 3;
                    na[0] = da[0]; na[1] = da[1]; na[2] = da[2];
                    nb[0] = da[96]; nb[1] = da[97]; nb[2] = da[98];
                }
                if (it > 0) {
                    mbar_wait(&s_done, (uint32_t)((it - 1) & 1));     // the transform has consumed the histogram
                    uint4 *h = reinterpret_cast<uint4 *>(smem + L.hist);
                    for (int i = bt; i < (int)(hist_bytes / 16); i += kBinThreads) h[i] = make_uint4(0, 0, 0, 0);
                    asm volatile("bar.sync 2, %0;" ::"n"(kBinThreads) : "memory");
                }
                const int a0 = pass * 2048, a1 = min(n, a0 + 2048);
                const int per = (a1 - a0 + kBinWarps - 1) / kBinWarps;
                const int i0 = min(a1, a0 + bw * per), i1 = min(a1, i0 + per);
                if (p.clamp) bin_ions<true>(ions_s, i0, i1, na, nb, c);
                else bin_ions<false>(ions_s, i0, i1, na, nb, c);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // histogram writes -> async proxy
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_full);
            }
        } else if (warp == kMmaWarp) {
            const uint32_t idesc = (1u << 4) | (1u << 15) | ((uint32_t)(p.N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
            const uint32_t tb = smem_u32(smem + L.table), hb = smem_u32(smem + L.hist);
            const uint32_t pair_off = (uint32_t)kRowGroupBytes * (uint32_t)(p.B / 16);
            for (int it = 0; it < nitems; ++it) {
                const int pass = it % npass;
                mbar_wait(&s_full, (uint32_t)(it & 1));
                if (it > 0) mbar_wait(&s_tfree, (uint32_t)((it - 1) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;");
                if (lane == 0) {
                    for (int pr = 0; pr < 2; ++pr)
                        for (int ks = 0; ks < K / 16; ++ks) {
                            uint64_t ad = make_desc(hb + pr * pair_off + ks * (4 * kRowGroupBytes), 2 * kRowGroupBytes, kChunkBytes, 0);
                            uint64_t bd = make_desc(tb + (ks >> 2) * p.N * 128 + (ks & 3) * 32, 16, 1024, 2);
                            mma_f16_ss(tmem + (uint32_t)(pr * p.N), ad, bd, idesc, (ks > 0 || pass > 0) ? 1u : 0u);
                        }
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                 ::"r"(smem_u32(&s_done)) : "memory");
                }
                __syncwarp();
            }
        } else {
            // ---- epilogue warps 0..3: TMEM lane = 32*warp + lane = M row blk*64 + slot --------------------
            const int blk = warp >> 1;
            const int et = (warp & 1) * 32 + lane;                                    // thread index among the 64 of this blk
            const int slot = ((lane & 1) << 5) + ((warp & 1) << 4) + ((lane >> 3) << 2) + ((lane & 7) >> 1);
            const uint32_t acc0 = tmem + ((uint32_t)(warp * 32) << 16);
            for (int it = 0; it < nitems; ++it) {
                const int gi = g_begin + it / npass;
                const bool last_pass = (it % npass) == npass - 1;
                mbar_wait(&s_done, (uint32_t)(it & 1));
                asm volatile("tcgen05.fence::after_thread_sync;");
                if (last_pass && blk == 0) asm volatile("bar.sync 1, 128;" ::: "memory");     // partner's partials are in exch
                float best = -1.0f;
                int kbest = p.k_lo;
                if (last_pass) {
#pragma unroll 1
                    for (int c = 0; c < p.N / 16; ++c) {
                        uint32_t v0[16], v1[16];
                        tmem_ld16(acc0 + (uint32_t)(c * 16), v0);
                        tmem_ld16(acc0 + (uint32_t)(p.N + c * 16), v1);
                        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int w = c * 4 + j;
                            if (w < p.W) {
                                const float r0 = __uint_as_float(v0[4 * j]) + __uint_as_float(v0[4 * j + 2]) * (1.0f / 2048.0f);
                                const float i0 = -(__uint_as_float(v0[4 * j + 1]) + __uint_as_float(v0[4 * j + 3]) * (1.0f / 2048.0f));
                                const float r1 = __uint_as_float(v1[4 * j]) + __uint_as_float(v1[4 * j + 2]) * (1.0f / 2048.0f);
                                const float i1 = -(__uint_as_float(v1[4 * j + 1]) + __uint_as_float(v1[4 * j + 3]) * (1.0f / 2048.0f));
                                const float2 f0 = phase[blk * p.W + w], f1 = phase[(2 + blk) * p.W + w];
                                float xr = (f0.x * r0 - f0.y * i0) + (f1.x * r1 - f1.y * i1);
                                float xi = (f0.x * i0 + f0.y * r0) + (f1.x * i1 + f1.y * r1);
                                if (blk == 1) {
                                    exch[w * 64 + et] = make_float2(xr, xi);
                                } else {
                                    const float2 o = exch[w * 64 + et];
                                    xr += o.x; xi += o.y;
                                    const float pw = xr * xr + xi * xi;
                                    if (pw > best) { best = pw; kbest = p.k_lo + w; }    // ascending w: lowest k kept on ties
                                }
                            }
                        }
                    }
                }
                // TMEM drained: the MMA warp may overwrite the accumulators
                asm volatile("tcgen05.fence::before_thread_sync;");
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_tfree);
                if (last_pass) {
                    if (blk == 1) {
                        asm volatile("bar.sync 1, 128;" ::: "memory");
                    } else {
                        const int d = p.perm[gi * 64 + slot];
                        if (d >= 0) p.sig[(size_t)m * p.D + d] = make_float2(16777216.0f * sqrtf(fmaxf(best, 0.0f)), (float)kbest);
                    }
                }
            }
        }
    }
    // ---- teardown ---------------------------------------------------------------------------------
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(p.tmem_cols));
}

// ---- host side ------------------------------------------------------------------------------------
static int mma_n_for(int W) { return ((4 * W + 15) / 16) * 16; }
static int mma_cap_for(int B, int N, int W)
{
    const int budget = 232448 - 512;   // 227 KB opt-in shared memory per CTA on sm_100, minus static shared
    MmaSmem s = mma_smem_layout(B, N, W, 0);
    int cap = ((budget - (int)s.total) / 16) & ~63;
    return cap > 4096 ? 4096 : cap;
}

bool mma_path_supported(const Plan *p)
{
    if (p->B > 1024) return false;                       // B = 2048, 4096 stay on the FFT kernel
    const int N = mma_n_for(p->W);
    if (2 * N > 512) return false;                       // two accumulators of N TMEM columns
    return mma_cap_for(p->B, N, p->W) >= 1024;           // room for a useful ion buffer
}

// Order the directions so that every run of 32 is a spatially compact patch: recursive bisection along the
// widest axis, cutting at a multiple of 32.  Within one shared atomic the 32 lanes then project an ion onto
// nearly parallel directions, their bins share the top three bits and the histogram layout is conflict-free.
static void patch_order(const std::vector<float> &v, std::vector<int> &idx, int lo, int hi)
{
    const int cnt = hi - lo;
    if (cnt <= 32) return;
    float mn[3] = {1e30f, 1e30f, 1e30f}, mx[3] = {-1e30f, -1e30f, -1e30f};
    for (int i = lo; i < hi; ++i)
        for (int a = 0; a < 3; ++a) {
            mn[a] = std::min(mn[a], v[3 * (size_t)idx[i] + a]);
            mx[a] = std::max(mx[a], v[3 * (size_t)idx[i] + a]);
        }
    int ax = 0;
    for (int a = 1; a < 3; ++a)
        if (mx[a] - mn[a] > mx[ax] - mn[ax]) ax = a;
    const int leaves = (cnt + 31) / 32;
    const int left = (leaves / 2) * 32;
    std::nth_element(idx.begin() + lo, idx.begin() + lo + left, idx.begin() + hi,
                     [&](int a, int b) { return v[3 * (size_t)a + ax] < v[3 * (size_t)b + ax]; });
    patch_order(v, idx, lo, lo + left);
    patch_order(v, idx, lo + left, hi);
}

cudaError_t mma_path_prepare(Plan *p)
{
    const int B = p->B, K = B / 4, W = p->W, N = mma_n_for(W);
    int nl = 0;
    while ((8 << nl) < B) ++nl;                          // B = 8 * 2^nl
    // twiddle table: K index k = kg*8 + hi3 stands for the bin part hi3*(B/8) + 2*kg
    std::vector<uint16_t> img((size_t)K * N, 0);
    for (int r = 0; r < K; ++r)
        for (int n = 0; n < N; ++n) {
            const int w = n / 4, c = n % 4;
            __half val = __float2half(0.0f);
            if (w < W) {
                const int64_t binpart = (int64_t)(r & 7) * (B / 8) + 2 * (r >> 3);
                const double th = 2.0 * M_PI * (double)((binpart * (p->k_lo + w)) % B) / (double)B;
                const double v = (c & 1) ? std::sin(th) : std::cos(th);
                const __half hi = __float2half((float)v);
                val = (c < 2) ? hi : __float2half((float)((v - (double)__half2float(hi)) * 2048.0));
            }
            // K-major SWIZZLE_128B image: k-block (64 rows of r) x [N rows of 128 B], 16-byte chunks XOR (n & 7)
            const size_t off = (size_t)(r / 64) * N * 64 + (size_t)n * 64 + (size_t)(((((r % 64) / 8) ^ (n % 8))) << 3) + (r % 8);
            img[off] = *reinterpret_cast<uint16_t *>(&val);
        }
    cudaError_t e = cudaMalloc(&p->d_mma_table, img.size() * 2);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p->d_mma_table, img.data(), img.size() * 2, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    // recombination phases exp(-2 pi i (pair*B/16 + blk) k / B)
    std::vector<float2> ph((size_t)4 * W);
    for (int pb = 0; pb < 4; ++pb)
        for (int w = 0; w < W; ++w) {
            const int64_t off = (int64_t)(pb >> 1) * (B / 16) + (pb & 1);
            const double th = 2.0 * M_PI * (double)((off * (p->k_lo + w)) % B) / (double)B;
            ph[(size_t)pb * W + w] = make_float2((float)std::cos(th), (float)-std::sin(th));
        }
    e = cudaMalloc(&p->d_mma_phase, ph.size() * sizeof(float2));
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p->d_mma_phase, ph.data(), ph.size() * sizeof(float2), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;

    std::vector<float> nps((size_t)3 * p->D);
    e = cudaMemcpy(nps.data(), p->d_dirs_scaled, nps.size() * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return e;
    // the clamp of Eq. 1's bin index can be skipped when it provably never triggers: paper padding
    // (pad = 1) and directions that are unit vectors to fp32 accuracy => |x| <= (B/2-1)(1+2e-5) < B/2 - 0.25
    bool unit = p->pad == 1;
    const double lim = (double)p->s * 1.00001;
    for (int d = 0; d < p->D && unit; ++d) {
        double nn = std::sqrt((double)nps[3 * d] * nps[3 * d] + (double)nps[3 * d + 1] * nps[3 * d + 1] +
                              (double)nps[3 * d + 2] * nps[3 * d + 2]);
        if (!(nn <= lim)) unit = false;
    }
    p->mma_clamp = unit ? 0 : 1;

    // patch order + padding to a multiple of 64 (padding slots repeat the last direction, perm = -1)
    std::vector<int> idx(p->D);
    std::iota(idx.begin(), idx.end(), 0);
    patch_order(nps, idx, 0, p->D);
    const int Dp = ((p->D + 63) / 64) * 64;
    std::vector<float> sorted((size_t)3 * Dp);
    std::vector<int> perm(Dp, -1);
    for (int i = 0; i < Dp; ++i) {
        const int src = idx[std::min(i, p->D - 1)];
        if (i < p->D) perm[i] = src;
        for (int a = 0; a < 3; ++a) sorted[3 * (size_t)i + a] = nps[3 * (size_t)src + a];
    }
    p->Dp = Dp;
    e = cudaMalloc(&p->d_dirs_sorted, sorted.size() * 4);
    if (e != cudaSuccess) return e;
    e = cudaMalloc(&p->d_dir_perm, perm.size() * 4);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p->d_dirs_sorted, sorted.data(), sorted.size() * 4, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    return cudaMemcpy(p->d_dir_perm, perm.data(), perm.size() * 4, cudaMemcpyHostToDevice);
}

cudaError_t launch_signature_mma(Plan *p, const float *centres, int64_t M, float *sig, uint32_t *counts, cudaStream_t st)
{
    if (M == 0) return cudaSuccess;
    // deferred list (material points whose ROI overflows the shared ion buffer), grown on demand
    if (M + 1 > p->cap_deferred) {
        if (p->d_deferred) cudaFree(p->d_deferred);
        p->d_deferred = nullptr; p->cap_deferred = 0;
        cudaError_t e = cudaMalloc(&p->d_deferred, (size_t)(M + 1) * 4);
        if (e != cudaSuccess) return e;
        p->cap_deferred = M + 1;
    }
    cudaError_t e = cudaMemsetAsync(p->d_deferred, 0, 4, st);
    if (e != cudaSuccess) return e;

    MmaParams q;
    q.sorted = p->d_sorted; q.cell_start = p->d_cell_start; q.grid = p->d_grid; q.centres = centres;
    q.dirs_sorted = p->d_dirs_sorted; q.perm = p->d_dir_perm;
    q.table = reinterpret_cast<const uint4 *>(p->d_mma_table); q.phase = p->d_mma_phase;
    q.sig = reinterpret_cast<float2 *>(sig); q.counts = counts; q.deferred = p->d_deferred;
    q.D = p->D; q.B = p->B; q.k_lo = p->k_lo; q.W = p->W; q.N = mma_n_for(p->W);
    q.nl = 0;
    while ((8 << q.nl) < p->B) ++q.nl;
    q.cap = mma_cap_for(p->B, q.N, p->W);
    q.ngroups = p->Dp / 64;
    int nchunks = (q.ngroups + 47) / 48;
    const int64_t want = (int64_t)p->sm_count * 8;
    if (M * nchunks < want) nchunks = (int)((want + M - 1) / M);
    if (nchunks > (q.ngroups + 1) / 2) nchunks = (q.ngroups + 1) / 2;
    if (nchunks < 1) nchunks = 1;
    q.nchunks = nchunks;
    q.clamp = p->mma_clamp;
    uint32_t cols = 32;
    while (cols < (uint32_t)(2 * q.N)) cols *= 2;
    q.tmem_cols = cols;
    q.R = p->R; q.R2 = p->R2;
    const MmaSmem L = mma_smem_layout(p->B, q.N, p->W, q.cap);
    e = cudaFuncSetAttribute(k_signature_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total);
    if (e != cudaSuccess) return e;
    const int64_t blocks = M * nchunks;
    if (blocks > 0x7FFFFFFFLL) return cudaErrorInvalidConfiguration;
    k_signature_mma<<<(unsigned)blocks, kMmaThreads, L.total, st>>>(q);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_signature_fft_list(p, centres, p->d_deferred, sig, counts, st);
}

}  // namespace apx
