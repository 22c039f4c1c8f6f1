// signature_mma.cu -- windowed-DFT signature kernel: shared-memory histograms feed the tcgen05 tensor
// cores directly (steps a2, a4-a7 for narrow spectral windows, B <= 1024).
//
// Per CTA: one material point x a chunk of direction groups (32 directions per group, lane = direction).
//   binning  : hist[b][32 dirs] u16 counters packed two directions per 32-bit word, updated with shared
//              atomics (Eq. 1).  The u16 bit pattern c is the fp16 number c * 2^-24
//              (subnormal / first binade, exact for c <= 2048), so the histogram IS a valid fp16
//              MN-major SWIZZLE_64B operand and is never converted or copied.
//   DFT      : X_k = sum_b h_b w^{bk} restricted to the window [k_lo,k_hi] is the dense contraction
//              [directions x bins] x [bins x window] (L73, L75).  With b = tau*K + r (tau = top 2 bits of
//              the bin, K = B/4) the four bin quarters become four M-blocks of one 128-row MMA tile and the
//              twiddle table shrinks to K x N: D[tau*32+d][n] = sum_r h[d][tau*K+r] T[r][n], then
//              X_k = sum_tau (-i)^{tau k} D_tau[k].  T holds cos/sin as fp16 hi + lo parts (columns
//              4w+{0,1,2,3} = cos_hi, sin_hi, 2^11 cos_lo, 2^11 sin_lo) so amplitudes reach ~1e-7 relative.
//   peak     : |X_k|^2 arg-max over the window, lowest k on ties (L75, L416); A* = 2^24 sqrt(max).
// Two histogram buffers and two TMEM accumulators: the tensor core transforms group g while the CUDA
// cores bin group g+1.  ROIs with more ions than the shared-memory ion buffer are appended to a
// deferred list and handled by the general FFT kernel.
#include <cmath>
#include <cuda_fp16.h>
#include <vector>
#include "common.cuh"

namespace apx {

constexpr int kBinWarps = 12;            // project-and-bin warps
constexpr int kMmaWarp = 4;              // tcgen05.mma issuer
constexpr int kFirstBinWarp = 5;         // warps 0..3 = epilogue (one per TMEM lane quarter)
constexpr int kMmaWarps = kFirstBinWarp + kBinWarps;
constexpr int kMmaThreads = kMmaWarps * 32;
constexpr int kIonBatch = 8;

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
// descriptor version 1, swizzle mode in bits 61-63 (2 = 128B, 4 = 64B)
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

struct MmaParams {
    const float4 *sorted;
    const uint32_t *cell_start;
    const GridParams *grid;
    const float *centres;
    const float *dirs_scaled;
    const uint4 *table;        // pre-swizzled twiddle operand image, (K/64) blocks of [N][128 B]
    float2 *sig;
    uint32_t *counts;
    uint32_t *deferred;        // [0] = count, [1..] = material point ids left to the FFT kernel
    int D, B, k_lo, W, N, cap, nchunks, ngroups, clamp;
    uint32_t tmem_cols;
    float R, R2;
};

// smem carve-up (bytes), shared by host and device
struct MmaSmem {
    uint32_t hist0, hist1, table, partial, best, ions, total;
};
__host__ __device__ inline MmaSmem mma_smem_layout(int B, int N, int W, int cap)
{
    MmaSmem s;
    uint32_t off = 0;
    s.hist0 = off; off += (uint32_t)B * 64;
    s.hist1 = off; off += (uint32_t)B * 64;
    s.table = off; off += (uint32_t)(B / 4) * N * 2;             // (K/64) * N * 128 with K = B/4
    s.partial = off; off += 4u * W * 32 * 8;
    s.best = off; off += kMmaWarps * 32 * 8;
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

// Project-and-bin (step a4) of ions [i0, i1) for this lane's direction into the SWIZZLE_64B histogram:
// byte offset of (bin b, direction lane) = b*64 + (((lane>>3) ^ ((b>>1)&3)) << 4) + ((lane&7)>>1)*4,
// low/high half of the word = even/odd lane.  With bits = 0x4B400000 + b (magic-add floor) this is
// addr = bits*64 + K0, then addr ^= (bits<<3) & 0x30.
__device__ __forceinline__ float4 lds128(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

template <bool kClamp>
__device__ __forceinline__ void bin_one(const float4 q, float npx, float npy, float npz, float half_b, float magic,
                                        uint32_t k0, uint32_t inc)
{
    float x = __fmaf_rn(npz, q.z, __fmaf_rn(npy, q.y, __fmul_rn(npx, q.x)));
    if (kClamp) x = fminf(fmaxf(x, -half_b), half_b - 0.25f);
    const uint32_t bits = __float_as_uint(__fadd_rd(x, magic));
    uint32_t addr = bits * 64u + k0;
    addr ^= (bits << 3) & 0x30u;
    red_shared_add(addr, inc);
}

// ions_s = shared-space byte address of the float4 ion records
template <bool kClamp>
__device__ __forceinline__ void bin_ions(uint32_t ions_s, int i0, int i1, float npx, float npy, float npz,
                                         float half_b, float magic, uint32_t k0, uint32_t inc)
{
    int ib = i0;
    for (; ib + kIonBatch <= i1; ib += kIonBatch) {          // full batches: loads first, then 8 independent chains
        float4 q[kIonBatch];
#pragma unroll
        for (int u = 0; u < kIonBatch; ++u) q[u] = lds128(ions_s + (uint32_t)(ib + u) * 16u);
#pragma unroll
        for (int u = 0; u < kIonBatch; ++u) bin_one<kClamp>(q[u], npx, npy, npz, half_b, magic, k0, inc);
    }
    for (; ib < i1; ++ib) bin_one<kClamp>(lds128(ions_s + (uint32_t)ib * 16u), npx, npy, npz, half_b, magic, k0, inc);
}

__global__ void __launch_bounds__(kMmaThreads, 1) k_signature_mma(const MmaParams p)
{
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 1024-byte aligned, still shared-space
    const MmaSmem L = mma_smem_layout(p.B, p.N, p.W, p.cap);
    __shared__ uint64_t s_full[2], s_done[2], s_empty[2];
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
    float2 *partial = reinterpret_cast<float2 *>(smem + L.partial);
    float2 *bestbuf = reinterpret_cast<float2 *>(smem + L.best);
    const int K = p.B / 4;

    // ---- setup: barriers, TMEM, zero histograms, twiddle table, gather ------------------------------
    if (tid == 0) {
        for (int i = 0; i < 2; ++i) {
            mbar_init(&s_full[i], kBinWarps);
            mbar_init(&s_done[i], 1);
            mbar_init(&s_empty[i], 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;");
        s_n = 0;
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(p.tmem_cols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    {
        uint4 *h = reinterpret_cast<uint4 *>(smem + L.hist0);
        for (int i = tid; i < p.B * 8; i += kMmaThreads) h[i] = make_uint4(0, 0, 0, 0);      // both buffers
        uint4 *t = reinterpret_cast<uint4 *>(smem + L.table);
        for (int i = tid; i < K * p.N / 8; i += kMmaThreads) t[i] = p.table[i];
    }
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
        // Warp-specialised pipeline over items = (direction group, ion pass):
        //   binning warps : wait empty[buf] -> project-and-bin the item into hist[buf] -> arrive full[buf]
        //   MMA warp      : wait full[buf]  -> K/16 tcgen05.mma into acc[group&1] -> commit to done[buf]
        //   epilogue warps: wait done[buf]  -> clear hist[buf]; on the last pass read TMEM, combine the four
        //                    bin quarters, arg-max, store; arrive empty[buf]
        const int npass = n > 2048 ? (n + 2047) / 2048 : 1;          // fp16 counters are exact up to 2048
        const int nitems = (g_end - g_begin) * npass;
        if (warp >= kFirstBinWarp) {
            const int bw = warp - kFirstBinWarp;
            const float half_b = (float)(p.B / 2), magic = magic_for(p.B);
            const uint32_t inc = (lane & 1) ? 65536u : 1u;
            const uint32_t lane_off = (uint32_t)((lane >> 3) << 4) + (uint32_t)(((lane & 7) >> 1) << 2);
            const uint32_t ions_s = smem_u32(ions);
            int d = min(g_begin * 32 + lane, p.D - 1);
            float npx = p.dirs_scaled[3 * d], npy = p.dirs_scaled[3 * d + 1], npz = p.dirs_scaled[3 * d + 2];
            for (int it = 0; it < nitems; ++it) {
                const int pass = it % npass;
                // prefetch the next group's direction while this item is binned
                float nx2 = npx, ny2 = npy, nz2 = npz;
                if (pass == npass - 1 && it + 1 < nitems) {
                    const int d2 = min((g_begin + (it + 1) / npass) * 32 + lane, p.D - 1);
                    nx2 = p.dirs_scaled[3 * d2]; ny2 = p.dirs_scaled[3 * d2 + 1]; nz2 = p.dirs_scaled[3 * d2 + 2];
                }
                if (it >= 2) mbar_wait(&s_empty[it & 1], (uint32_t)(((it - 2) >> 1) & 1));
                const int a0 = pass * 2048, a1 = min(n, a0 + 2048);
                const int per = (a1 - a0 + kBinWarps - 1) / kBinWarps;
                const int i0 = min(a1, a0 + bw * per), i1 = min(a1, i0 + per);
                const uint32_t hb = smem_u32(smem + ((it & 1) ? L.hist1 : L.hist0));
                const uint32_t k0 = hb + lane_off - 0x4B400000u * 64u;
                if (p.clamp) bin_ions<true>(ions_s, i0, i1, npx, npy, npz, half_b, magic, k0, inc);
                else bin_ions<false>(ions_s, i0, i1, npx, npy, npz, half_b, magic, k0, inc);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // histogram writes -> async proxy
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_full[it & 1]);
                npx = nx2; npy = ny2; npz = nz2;
            }
        } else if (warp == kMmaWarp) {
            const uint32_t idesc = (1u << 4) | (1u << 15) | ((uint32_t)(p.N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
            const uint32_t tb = smem_u32(smem + L.table);
            for (int it = 0; it < nitems; ++it) {
                const int gi = g_begin + it / npass, pass = it % npass;
                mbar_wait(&s_full[it & 1], (uint32_t)((it >> 1) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;");
                if (lane == 0) {
                    const uint32_t acc = tmem + (uint32_t)((gi & 1) * p.N);
                    const uint32_t ha = smem_u32(smem + ((it & 1) ? L.hist1 : L.hist0));
                    for (int ks = 0; ks < K / 16; ++ks) {
                        uint64_t ad = make_desc(ha + ks * 1024, (uint32_t)K * 64, 512, 4);
                        uint64_t bd = make_desc(tb + (ks >> 2) * p.N * 128 + (ks & 3) * 32, 16, 1024, 2);
                        mma_f16_ss(acc, ad, bd, idesc, (ks > 0 || pass > 0) ? 1u : 0u);
                    }
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                 ::"r"(smem_u32(&s_done[it & 1])) : "memory");
                }
                __syncwarp();
            }
        } else {
            // ---- epilogue warps 0..3 (TMEM lane quarter = bin quarter tau = warp) -------------------------
            const int tau = warp, et = tid;                               // et in [0,128)
            for (int it = 0; it < nitems; ++it) {
                const int gp = g_begin + it / npass;
                const bool last_pass = (it % npass) == npass - 1;
                mbar_wait(&s_done[it & 1], (uint32_t)((it >> 1) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;");
                {   // the transform has consumed this histogram: clear it for item it+2
                    uint4 *h = reinterpret_cast<uint4 *>(smem + ((it & 1) ? L.hist1 : L.hist0));
                    for (int i = et; i < p.B * 4; i += 128) h[i] = make_uint4(0, 0, 0, 0);
                }
                if (last_pass) {
                    const uint32_t acc = tmem + (uint32_t)((gp & 1) * p.N) + ((uint32_t)(tau * 32) << 16);
                    for (int c = 0; c < p.N / 16; ++c) {
                        uint32_t v[16];
                        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                                       "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                                     : "r"(acc + (uint32_t)(c * 16)));
                        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int w = c * 4 + j;
                            if (w < p.W) {
                                float re = __uint_as_float(v[4 * j]) + __uint_as_float(v[4 * j + 2]) * (1.0f / 2048.0f);
                                float im = -(__uint_as_float(v[4 * j + 1]) + __uint_as_float(v[4 * j + 3]) * (1.0f / 2048.0f));
                                const int e = (tau * (p.k_lo + w)) & 3;             // (-i)^(tau k)
                                float xr = (e == 0) ? re : (e == 1) ? im : (e == 2) ? -re : -im;
                                float xi = (e == 0) ? im : (e == 1) ? -re : (e == 2) ? -im : re;
                                partial[(tau * p.W + w) * 32 + lane] = make_float2(xr, xi);
                            }
                        }
                    }
                }
                // histogram cleared and TMEM drained: hand the buffer (and accumulator) back
                asm volatile("tcgen05.fence::before_thread_sync;");
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_empty[it & 1]);
                if (last_pass) {
                    asm volatile("bar.sync 1, 128;" ::: "memory");
                    float best = -1.0f;
                    int kbest = p.k_lo;
                    for (int w = warp; w < p.W; w += 4) {
                        float2 a = partial[(0 * p.W + w) * 32 + lane], b = partial[(1 * p.W + w) * 32 + lane];
                        float2 c2 = partial[(2 * p.W + w) * 32 + lane], d2 = partial[(3 * p.W + w) * 32 + lane];
                        float xr = (a.x + b.x) + (c2.x + d2.x), xi = (a.y + b.y) + (c2.y + d2.y);
                        float pw = xr * xr + xi * xi;
                        if (pw > best) { best = pw; kbest = p.k_lo + w; }
                    }
                    bestbuf[warp * 32 + lane] = make_float2(best, __int_as_float(kbest));
                    asm volatile("bar.sync 1, 128;" ::: "memory");
                    if (warp == 0) {
                        float bb = -1.0f;
                        int kb = p.k_lo;
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            float2 c = bestbuf[j * 32 + lane];
                            int ck = __float_as_int(c.y);
                            if (c.x > bb || (c.x == bb && ck < kb)) { bb = c.x; kb = ck; }
                        }
                        const int dg = gp * 32 + lane;
                        if (dg < p.D)
                            p.sig[(size_t)m * p.D + dg] = make_float2(16777216.0f * sqrtf(fmaxf(bb, 0.0f)), (float)kb);
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
    if (N > 256) return false;
    return mma_cap_for(p->B, N, p->W) >= 1024;           // room for a useful ion buffer
}

cudaError_t mma_path_prepare(Plan *p)
{
    const int B = p->B, K = B / 4, W = p->W, N = mma_n_for(W);
    std::vector<uint16_t> img((size_t)K * N, 0);
    for (int r = 0; r < K; ++r)
        for (int n = 0; n < N; ++n) {
            const int w = n / 4, c = n % 4;
            __half val = __float2half(0.0f);
            if (w < W) {
                const double th = 2.0 * M_PI * (double)(((int64_t)r * (p->k_lo + w)) % B) / (double)B;
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
    // the clamp of Eq. 1's bin index can be skipped when it provably never triggers: paper padding
    // (pad = 1) and directions that are unit vectors to fp32 accuracy => |x| <= (B/2-1)(1+2e-5) < B/2 - 0.25
    std::vector<float> nps((size_t)3 * p->D);
    e = cudaMemcpy(nps.data(), p->d_dirs_scaled, nps.size() * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return e;
    bool unit = p->pad == 1;
    const double lim = (double)p->s * 1.00001;
    for (int d = 0; d < p->D && unit; ++d) {
        double nn = std::sqrt((double)nps[3 * d] * nps[3 * d] + (double)nps[3 * d + 1] * nps[3 * d + 1] +
                              (double)nps[3 * d + 2] * nps[3 * d + 2]);
        if (!(nn <= lim)) unit = false;
    }
    p->mma_clamp = unit ? 0 : 1;
    return cudaSuccess;
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
    q.dirs_scaled = p->d_dirs_scaled; q.table = reinterpret_cast<const uint4 *>(p->d_mma_table);
    q.sig = reinterpret_cast<float2 *>(sig); q.counts = counts; q.deferred = p->d_deferred;
    q.D = p->D; q.B = p->B; q.k_lo = p->k_lo; q.W = p->W; q.N = mma_n_for(p->W);
    q.cap = mma_cap_for(p->B, q.N, p->W);
    q.ngroups = (p->D + 31) / 32;
    int nchunks = (q.ngroups + 47) / 48;
    const int64_t want = (int64_t)p->sm_count * 8;
    if (M * nchunks < want) nchunks = (int)((want + M - 1) / M);
    if (nchunks > (q.ngroups + 3) / 4) nchunks = (q.ngroups + 3) / 4;
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
