// signature_mma.cu -- windowed-DFT signature kernel: shared-memory histograms feed the tcgen05 tensor
// cores directly (steps a2, a4-a7 for narrow spectral windows, B <= 2048).
//
// Per CTA: one material point x a chunk of direction groups; a group = G direction slots (32 for B <= 1024, 16 for
// B = 2048; struct Lay).  Described for B = 1024:
//   binning  : lane l (0..15) of a half-warp owns ONE 32-bit word per histogram row: two u16 counters, the
//              low half for direction l (set A) and the high half for direction l + 16 (set B) of the group
//              (Eq. 1).  The two half-warps of a warp work on different ions, every lane bins its
//              ions for both of its directions.  The u16 bit pattern c is the fp16 number c * 2^-24 (subnormal /
//              first binade, exact for c <= 2048), so the histogram IS a valid fp16 tensor-core operand and is never
//              converted or copied.
//   layout   : byte address of (bin b, lane l) = (l/4)*160 + (l%4)*4 + 16*hi3 + 640*low,
//              hi3 = b >> (log2 B - 3), low = b & (B/8 - 1).  Bank = 8*(l/4) + 4*hi3 + l%4 (mod 32): the 16 lanes
//              of a half-warp hit 16 different banks whenever their bins agree in the top three bits (hi3) -- the
//              plan sorts the directions into spatially compact patches of 16 so that they almost always do --
//              and the other half-warp falls on the other 16 banks when its hi3 has the other parity.
//              Read as an MN-major INTERLEAVE (no swizzle) operand with SBO = 160 B (between 8-element M chunks)
//              and LBO = 2560 B (between 8-row K groups) this is a [128 x K] tile: M row = blk*32 + direction slot
//              (blk = low & 3), K index = kg*8 + hi3 (kg = low >> 2), K = B/4.
//   DFT      : X_k = sum_b h_b w^{bk} restricted to the window [k_lo,k_hi] is the dense contraction
//              [directions x bins] x [bins x window] (L73, L75).  With b = hi3*B/8 + 4*kg + blk the four blk parts
//              share one twiddle table T[k=(kg,hi3)][n] and are recombined in the epilogue with the phases
//              w^{blk k}.  T holds cos/sin as fp16 hi + lo parts (columns 4w+{0,1,2,3} = cos_hi, sin_hi,
//              2^11 cos_lo, 2^11 sin_lo) so amplitudes reach ~1e-7.
//   peak     : |X_k|^2 arg-max over the window, lowest k on ties (L75, L416); A* = 2^24 sqrt(max).
// Two histogram buffers and two TMEM accumulators: while the 16 binning warps fill buffer (g+1)&1, the tensor
// core transforms buffer g&1, a TMA bulk copy clears it and one of two sets of four service warps runs the epilogue
// of group g.  A ROI with more ions than the ion buffer spills into the second histogram buffer and runs
// single-buffered (so does every ROI at B = 2048, where only one buffer fits); only ROIs beyond that are appended to
// a deferred list for the general FFT kernel.
// Half-grid mode (antipodally symmetric direction grids, L60): one member of every pair (n, -n) is binned and its peak
// serves both; see the comment above struct Detect.
#include <algorithm>
#include <array>
#include <cstdlib>
#include <cstring>
#include <map>
#include <cmath>
#include <cuda_fp16.h>
#include <numeric>
#include <type_traits>
#include <vector>
#include "common.cuh"

namespace apx {

constexpr int kBinWarps = 16;            // warps 0..15: project-and-bin
constexpr int kMmaWarp = 16;             // tcgen05.mma issuer
constexpr int kClrWarp = 17;             // issues the TMA bulk clears
constexpr int kSvcWarp0 = 18;            // warps 18..25: epilogue (TMEM quarter = warp & 3),
constexpr int kSvcWarps = 8;             // two sets of four warps; set s takes the groups with (group & 1) == s
constexpr int kMmaWarps = kSvcWarp0 + kSvcWarps;
constexpr int kMmaThreads = kMmaWarps * 32;
// Histogram layout, by the number NB of bin parts that sit side by side in the M dimension of the tensor-core operand:
// b = hi3 * B/8 + NB * kg + blk (blk < NB), M row = blk * G + direction slot, K index = kg * 8 + hi3, K = B / NB.
//   NB = 4 (B <= 1024): G = 32 slots per group, 16 words per histogram row, two ion streams (half-warps) per warp
//   NB = 8 (B = 2048) : G = 16 slots per group,  8 words per histogram row, four ion streams (quarter-warps) per warp
// SBO (bytes between 8-slot M chunks) = 128 + a skew that puts the words of a row on different banks for a common hi3
// and keeps the stride of `low` (= BLK) a multiple of 128 B, i.e. bank neutral; LBO = 16 M chunks = one 8-row K group.
template <int NB>
struct Lay {
    static constexpr int G = 128 / NB;
    static constexpr int LW = G / 2;                 // lanes per ion stream = words per histogram row
    static constexpr int NS = 32 / LW;               // ion streams per warp
    static constexpr int SBO = NB == 4 ? 160 : 192;
    static constexpr int BLK = (G / 8) * SBO;        // one (blk, kg) slab: 640 / 384 B
    static constexpr int LBO = 16 * SBO;             // 2560 / 3072 B
};
__host__ __device__ inline int mma_nb_for(int B) { return B > 1024 ? 8 : 4; }
__host__ __device__ inline int mma_sbo_for(int nb) { return nb == 4 ? 160 : 192; }
constexpr int kStsClearBelow = 700;      // ROIs with fewer ions clear with plain stores instead of TMA copies from L2
constexpr int kEpiRound = 4;             // window bins per epilogue round (one tcgen05.ld x16)

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// Development aid (build with -DAPX_TRACE): lane 0 of selected warps of ONE CTA appends (event, group, SM clock) records to a
// global buffer, which shows the timeline of the warp-specialised pipeline.  Compiled out otherwise.
#ifdef APX_TRACE
// per-warp regions of trace_cap records each, index kept in a register (trace_n of run_pipeline): two plain stores per
// event, no atomics, nothing to wait for -- the timeline is not disturbed
#define APX_TRACE_EVENT(p, ev, grp)                                                                   \
    do {                                                                                              \
        if ((p).trace && blockIdx.x == (unsigned)(p).trace_block && (threadIdx.x & 31) == 0 && trace_n < (p).trace_cap) { \
            long long *r__ = (p).trace + 2 * ((long long)(threadIdx.x >> 5) * (p).trace_cap + trace_n++);       \
            r__[0] = ((long long)(ev) << 48) | ((long long)(threadIdx.x >> 5) << 32) | (long long)(grp) | (1ll << 62); \
            r__[1] = clock64();                                                                       \
        }                                                                                             \
    } while (0)
#else
#define APX_TRACE_EVENT(p, ev, grp) do { } while (0)
#endif
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t cnt)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(cnt));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(smem_u32(bar)) : "memory");
}
template <unsigned kSleepNs = 64>
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    uint32_t spins = 0;
    do {
        // the hint lets the hardware park the warp (up to ~1 ms) instead of burning issue slots in a spin loop
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity), "r"(1000000u) : "memory");
        if (!done) {
            __nanosleep(kSleepNs);                                   // do not burn issue slots of the binning warps
            if (++spins > (1u << 22)) asm volatile("trap;");         // never hang the device on a lost commit
        }
    } while (!done);
}
// The same wait as one tight PTX loop (no flag materialised in a register, no selp), for the two waits that poll most
// (binning warps on `free`, service warps on `epi`).  It carries the same guard: after 2^22 unsuccessful attempts (seconds)
// the warp traps instead of hanging the device on a lost arrival.
template <unsigned kSleepNs = 64>
__device__ __forceinline__ void mbar_wait_lean(uint64_t *bar, uint32_t parity)
{
    asm volatile("{\n .reg .pred p;\n .reg .u32 n;\n mov.u32 n, 0;\n"
                 "WAIT_LOOP:\n"
                 " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
                 " @p bra WAIT_DONE;\n"
                 " nanosleep.u32 %3;\n"
#ifndef APX_LEAN_NOGUARD
                 " add.u32 n, n, 1;\n"
                 " setp.gt.u32 p, n, 4194304;\n"
                 " @p trap;\n"
#endif
                 " bra WAIT_LOOP;\n"
                 "WAIT_DONE:\n}"
                 ::"r"(smem_u32(bar)), "r"(parity), "r"(1000000u), "n"(kSleepNs) : "memory");
}
__device__ __forceinline__ void mma_f16_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc)
{
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_f16_acc(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc)
{
    asm volatile("{\n .reg .pred p;\n setp.eq.b32 p, 0, 0;\n tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc) : "memory");
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

__device__ __forceinline__ uint32_t tmem_ld1(uint32_t addr)
{
    uint32_t v;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

struct MmaParams {
    const float4 *sorted;
    const uint32_t *cell_start;
    const GridParams *grid;
    const float *centres;
    const float *dirs_sorted;  // [Dp][3] scaled directions in patch order (Dp = D rounded up to 32)
    const int *perm;           // [Dp] original direction index of each sorted slot, -1 = padding
    const int *perm_mirror;    // [Dp] half-grid mode: index of the direction opposite to the slot's, else nullptr
    const uint4 *table;        // pre-swizzled twiddle operand image, (K/64) blocks of [N][128 B]
    const float2 *phase;       // [4][W] recombination phases w^{blk k}
    const void *zeros;         // hist_bytes of zeros: source of the bulk copies that clear a histogram buffer
    float2 *sig;
    uint32_t *counts;
    uint32_t *deferred;        // [0] = count, [1..] = material point ids left to the FFT kernel
    uint32_t *hist_out;        // test hook (apx_debug_histograms, M = 1): uint32[hist_nd][B] histograms of the directions
    int hist_d0, hist_nd;      // [hist_d0, hist_d0 + hist_nd), decoded from the shared-memory buffers the tensor core reads
#ifdef APX_TRACE
    long long *trace;          // [0] = record count, then (tag, clock) pairs
    int trace_block, trace_cap;
#endif
    int D, B, nl, k_lo, W, N, cap, cap_big, nchunks, ngroups, clamp, M;
    int half;                  // 1 = half-grid mode: one direction per antipodal pair is binned (perm_mirror != nullptr)
    int norm0;                 // single-signature plans: 1 = write A / N_c
    SpecSet ss;                // signatures of the plan: classes (type masks), per-spec sub-windows of [k_lo, k_lo + W)
    int nacc, nacc_log2;       // TMEM accumulators (2 or 4): group gq uses accumulator gq & (nacc - 1), so the MMAs of a group
                               // wait for the epilogue of group gq - nacc only
    int dc_col;                // >= 0: spare accumulator column 4 W whose twiddle is 1 for every bin: it receives the sum of the
                               // counters AS THE TENSOR CORE READ THEM, = N_c exactly unless a counter exceeded 2048 (see pass_ions)
    int pass_ions;             // ions binned per pass: 2048 (no counter can leave the exactly aliased range), or, with dc_col,
                               // the whole ROI in one pass, checked after the fact by the DC column
    int unit_split;            // 1 = ions are dealt to the binning warps in whole blocks of 4 * NS (no ragged tails)
    uint32_t tmem_cols;
    float R, R2;
};

// smem carve-up (bytes), shared by host and device
struct MmaSmem {
    uint32_t table, hist0, hist1, exch, cand, phase, ions, hist_bytes, total;
};
__host__ __device__ inline MmaSmem mma_smem_layout(int B, int N, int W, int cap)
{
    MmaSmem s;
    uint32_t off = 0;
    const int nb = mma_nb_for(B), K = B / nb;
    s.hist_bytes = (uint32_t)(K / 8) * 16u * (uint32_t)mma_sbo_for(nb);   // K/8 K groups of LBO bytes
    s.table = off; off += (uint32_t)K * N * 2;                   // (K/64) * N * 128; multiple of 1024
    s.hist0 = off; off += s.hist_bytes;
    s.exch = off; off += 2u * kEpiRound * 4 * 32 * 8;             // per set, one epilogue round: 4 bins x 4 warps x 32 lanes x float2
    s.cand = off; off += 8u * 32 * 8;
    s.phase = off; off += (uint32_t)nb * W * 8;
    s.ions = off; off += (uint32_t)cap * 12;
    if (nb == 4) {
        s.hist1 = off; off += s.hist_bytes;                        // directly behind the ion buffer: a ROI with more than
                                                                   // `cap` ions spills into it and runs single-buffered
    } else {
        s.hist1 = s.hist0;                                         // B = 2048: room for one histogram buffer only
    }
    s.total = off + 1024;                                          // slack for 1024-byte alignment
    return s;
}

// Gather (step a2) into quad-blocked records: four ions = 48 B = [dx0..dx3][dy0..dy3][dz0..dz3], i.e. three LDS.128
// whose register pairs are the operands of the packed fp32x2 arithmetic of the binning warps.
template <bool kMulti>
__device__ __forceinline__ void gather_roi3(const MmaParams &p, const GridParams &g, const RoiCells &rc,
                                            float cx, float cy, float cz, float *ions, int *s_n, int cls, int nwarps)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;     // warps 0 .. nwarps-1 gather
    const int ny_r = rc.iy1 - rc.iy0 + 1, nz_r = rc.iz1 - rc.iz0 + 1;
    for (int row = wid; row < ny_r * nz_r; row += nwarps) {
        int iy = rc.iy0 + row % ny_r, iz = rc.iz0 + row / ny_r;
        int base = (iz * g.ny + iy) * g.nx;
        uint32_t beg = p.cell_start[base + rc.ix0], end = p.cell_start[base + rc.ix1 + 1];
        for (uint32_t i = beg + lane; i < ((end - beg + 31u) & ~31u) + beg; i += 32) {
            bool in = false;
            float dx = 0.f, dy = 0.f, dz = 0.f;
            if (i < end) {
                float4 q = p.sorted[i];
                dx = __fsub_rn(q.x, cx); dy = __fsub_rn(q.y, cy); dz = __fsub_rn(q.z, cz);
                in = inside(dx, dy, dz, p.R2) && (!kMulti || p.ss.n_classes == 1 || type_in_class(p.ss, cls, __float_as_uint(q.w)));
            }
            unsigned msk = __ballot_sync(0xffffffffu, in);
            if (msk) {
                int pos = 0;
                if (lane == 0) pos = atomicAdd(s_n, __popc(msk));
                pos = __shfl_sync(0xffffffffu, pos, 0) + __popc(msk & ((1u << lane) - 1u));
                if (in && pos < p.cap_big) {                   // quad-blocked: [x0..x3][y0..y3][z0..z3] per four ions
                    float *q = ions + (pos >> 2) * 12 + (pos & 3);
                    q[0] = dx; q[4] = dy; q[8] = dz;
                }
            }
        }
    }
}

// Project-and-bin (step a4).  Lane (h = lane >> 4, l = lane & 15) owns word l of every histogram row: the low u16 is
// direction l of set A (increment 1), the high u16 direction l of set B (increment 65536).  The two half-warps take
// alternate blocks of the warp's ions and every lane bins each of its ions for BOTH of its directions, so one ion
// load (broadcast LDS.128, 2.2 clk on B200 whether the half-warps read the same or different addresses) serves two
// (ion, direction) pairs.  The plan pairs every compact patch A with the patch B nearest to its antipode.
//   ua = bits(RD(x + 1.5*2^23 + B/2))       = 0x4B400000 + b          (b = B/2 + floor(x), Eq. 1)
//   va = bits(RD(x*2^-nl + 1.5*2^23 + 4))   = 0x4B400000 + hi3        (hi3 = b >> nl, exact: floor(floor(y)/n) = floor(y/n))
//   address = hist + lane offset + 640*low + 16*hi3 = ua*640 + va*(16 - 640*2^nl) + k0   (mod 2^32)
// Two ions are projected at once with the packed fp32x2 instructions of sm_100 (FMUL2 / FFMA2 / FADD2.RM /
// FFMA2.RM: IEEE single roundings per component, same operation order as the contract): 5 packed + 2 x (2 IMAD +
// ATOMS) = 5.5 issue slots per (ion, direction) pair instead of 8.
struct BinConst {
    float half_b, magic_a, magic_b, scl;
    uint32_t kz;
};
__device__ __forceinline__ uint64_t pack2(float lo, float hi)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
template <bool kClamp, bool kDetect, int BLK>
__device__ __forceinline__ bool bin_one(float dx, float dy, float dz, float npx, float npy, float npz, const BinConst &c,
                                        uint32_t k0, uint32_t inc)
{
    float x = __fmaf_rn(npz, dz, __fmaf_rn(npy, dy, __fmul_rn(npx, dx)));
    if (kClamp) x = fminf(fmaxf(x, -c.half_b), c.half_b - 0.25f);
    const uint32_t ua = __float_as_uint(__fadd_rd(x, c.magic_a));
    const uint32_t va = __float_as_uint(__fmaf_rd(x, c.scl, c.magic_b));
    red_shared_add(ua * (uint32_t)BLK + (va * c.kz + k0), inc);
    return kDetect && ua == __float_as_uint(__fadd_ru(x, c.magic_a));      // true: x is an exact integer
}
// Half-grid mode (antipodally symmetric direction grids such as the geodesic mesh of the paper, L60): only one
// direction v of every pair (v, -v) is binned.  x(-v) = -x(v) bit for bit (every product and sum is negated exactly), so
// b(-v) = B/2 + floor(-x) = B - 1 - b(v) whenever x is not an integer: the histogram of -v is the mirror image of the
// histogram of v and has the same amplitude spectrum.  x is an integer exactly when rounding x + magic down and up gives
// the same number; a pair for which that happens for any ion (~1e-5 of all (ion, direction) pairs) is flagged, its -v
// member gets no output from this group and is binned on its own in a fix-up group.
// flag words in flight: the binning warps run at most nacc + 1 groups ahead of the epilogue that reads and resets a group's
// word (bin(g + nacc + 2) needs the buffer back from the MMAs of g + nacc, which wait for the epilogue of g): 8 slots for up to
// four accumulators
constexpr int kFlagSlots = 8;
constexpr int kFixCap = 512;             // flagged pairs per sub-range of kSubGroups groups
constexpr int kSubGroups = 128;
// Shared state of the flagging: one struct so that the rarely-taken path needs one base address.
struct FixShared {
    uint32_t flag[kFlagSlots];           // flag word per group in flight: bit s = slot s has met an exact-integer projection
    int nfix;                            // number of listed pairs of the sub-range
    uint16_t fix[kFixCap];               // flagged pairs: (group within the sub-range) * G + slot
};
// What a binning lane needs to flag one of its two pairs -- two registers, opaque to the compiler (it would otherwise
// re-derive the addresses from the thread id and the shared-memory window inside the hot loop):
//   base_s = shared-space address of the FixShared; ctx = flag slot | lane word l << 4 | (group within sub-range * G) << 16
struct Detect {
    uint32_t base_s, ctx;
};
// set = 0: the lane's set-A direction (slot l), 1: its set-B direction (slot LW + l)
template <int LW>
__device__ __noinline__ void flag_pair(uint32_t base_s, uint32_t ctx, uint32_t set)
{
    const uint32_t slot = ((ctx >> 4) & 0xFFFu) + set * (uint32_t)LW, bit = 1u << slot, id = (ctx >> 16) + slot;
    uint32_t old;
    asm volatile("atom.shared.or.b32 %0, [%1], %2;" : "=r"(old) : "r"(base_s + 4u * (ctx & 15u)), "r"(bit) : "memory");
    if (!(old & bit)) {
        uint32_t i;
        asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(i) : "r"(base_s + (uint32_t)offsetof(FixShared, nfix)) : "memory");
        if (i < (uint32_t)kFixCap)
            asm volatile("st.shared.u16 [%0], %1;" ::"r"(base_s + (uint32_t)offsetof(FixShared, fix) + 2u * i), "h"((uint16_t)id) : "memory");
    }
}
// two ions (dx0,dx1), (dy0,dy1), (dz0,dz1) for this lane's direction
// kDetect: nonint accumulates the number of the projections that are NOT exact integers: the bit patterns of RU(x + magic)
// and RD(x + magic) differ by exactly 1 for a non-integer x and by 0 for an integer.  (A packed-FP variant of the count --
// FADD2.RP, packed subtract, packed add -- was measured slower: it moves work to the FMA pipe the projections already load.)
template <bool kDetect, int BLK>
__device__ __forceinline__ void bin_pair(float dx0, float dx1, float dy0, float dy1, float dz0, float dz1, uint64_t nx2,
                                         uint64_t ny2, uint64_t nz2, uint64_t ma2, uint64_t sc2, uint64_t mb2, uint32_t kz,
                                         uint32_t k0, uint32_t inc, uint32_t &nonint)
{
    uint64_t t, ua, va;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(t) : "l"(nx2), "l"(pack2(dx0, dx1)));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(t) : "l"(ny2), "l"(pack2(dy0, dy1)), "l"(t));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(t) : "l"(nz2), "l"(pack2(dz0, dz1)), "l"(t));
    asm("add.rm.f32x2 %0, %1, %2;" : "=l"(ua) : "l"(t), "l"(ma2));
    asm("fma.rm.f32x2 %0, %1, %2, %3;" : "=l"(va) : "l"(t), "l"(sc2), "l"(mb2));
    const uint32_t ua0 = (uint32_t)ua, ua1 = (uint32_t)(ua >> 32), va0 = (uint32_t)va, va1 = (uint32_t)(va >> 32);
    red_shared_add(ua0 * (uint32_t)BLK + (va0 * kz + k0), inc);
    red_shared_add(ua1 * (uint32_t)BLK + (va1 * kz + k0), inc);
    if (kDetect) {
        uint64_t up;
        asm("add.rp.f32x2 %0, %1, %2;" : "=l"(up) : "l"(t), "l"(ma2));
        nonint += ((uint32_t)up - ua0) + ((uint32_t)(up >> 32) - ua1);
    }
}

// One direction pair of a lane: set A (low u16, increment 1) and set B (high u16, increment 65536) of the same word.
struct LaneDirs {
    float ax, ay, az, bx, by, bz;
};
// ions_s = shared-space byte address of the quad-blocked ion records; i0 is a multiple of 4.  The two half-warps of a
// warp take alternate blocks of ions (half h = lane >> 4), every lane bins each of its ions for BOTH of its directions,
// so one ion load serves two (ion, direction) pairs.
template <bool kClamp, bool kDetect, int NB>
__device__ __forceinline__ void bin_ions(uint32_t ions_s, int i0, int i1, const LaneDirs &n, const BinConst &c, uint32_t k0,
                                         int h, const Detect &dt)
{
    constexpr int NS = Lay<NB>::NS, BLK = Lay<NB>::BLK;
    int ib = i0;
    if (!kClamp) {
        const uint64_t ax2 = pack2(n.ax, n.ax), ay2 = pack2(n.ay, n.ay), az2 = pack2(n.az, n.az);
        const uint64_t bx2 = pack2(n.bx, n.bx), by2 = pack2(n.by, n.by), bz2 = pack2(n.bz, n.bz);
        const uint64_t ma2 = pack2(c.magic_a, c.magic_a), sc2 = pack2(c.scl, c.scl), mb2 = pack2(c.magic_b, c.magic_b);
        uint32_t src = ions_s + (uint32_t)ib * 12u + (uint32_t)h * 96u;
        for (; ib + 8 * NS <= i1; ib += 8 * NS, src += 96u * NS) {   // 8 ions per stream = 6 LDS.128, then 8 packed chains
            float4 q[6];
#pragma unroll
            for (int u = 0; u < 6; ++u) q[u] = lds128(src + (uint32_t)u * 16u);
            uint32_t na = 0u, nb = 0u;
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const float4 X = q[3 * hh], Y = q[3 * hh + 1], Z = q[3 * hh + 2];
                bin_pair<kDetect, BLK>(X.x, X.y, Y.x, Y.y, Z.x, Z.y, ax2, ay2, az2, ma2, sc2, mb2, c.kz, k0, 1u, na);
                bin_pair<kDetect, BLK>(X.z, X.w, Y.z, Y.w, Z.z, Z.w, ax2, ay2, az2, ma2, sc2, mb2, c.kz, k0, 1u, na);
                bin_pair<kDetect, BLK>(X.x, X.y, Y.x, Y.y, Z.x, Z.y, bx2, by2, bz2, ma2, sc2, mb2, c.kz, k0, 65536u, nb);
                bin_pair<kDetect, BLK>(X.z, X.w, Y.z, Y.w, Z.z, Z.w, bx2, by2, bz2, ma2, sc2, mb2, c.kz, k0, 65536u, nb);
            }
            if (kDetect) {
                if (__builtin_expect(na != 8u, 0)) flag_pair<Lay<NB>::LW>(dt.base_s, dt.ctx, 0u);
                if (__builtin_expect(nb != 8u, 0)) flag_pair<Lay<NB>::LW>(dt.base_s, dt.ctx, 1u);
            }
        }
        if (ib + 4 * NS <= i1) {                             // one quad per stream
            const uint32_t a = ions_s + (uint32_t)ib * 12u + (uint32_t)h * 48u;
            const float4 X = lds128(a), Y = lds128(a + 16u), Z = lds128(a + 32u);
            uint32_t na = 0u, nb = 0u;
            bin_pair<kDetect, BLK>(X.x, X.y, Y.x, Y.y, Z.x, Z.y, ax2, ay2, az2, ma2, sc2, mb2, c.kz, k0, 1u, na);
            bin_pair<kDetect, BLK>(X.z, X.w, Y.z, Y.w, Z.z, Z.w, ax2, ay2, az2, ma2, sc2, mb2, c.kz, k0, 1u, na);
            bin_pair<kDetect, BLK>(X.x, X.y, Y.x, Y.y, Z.x, Z.y, bx2, by2, bz2, ma2, sc2, mb2, c.kz, k0, 65536u, nb);
            bin_pair<kDetect, BLK>(X.z, X.w, Y.z, Y.w, Z.z, Z.w, bx2, by2, bz2, ma2, sc2, mb2, c.kz, k0, 65536u, nb);
            if (kDetect) {
                if (__builtin_expect(na != 4u, 0)) flag_pair<Lay<NB>::LW>(dt.base_s, dt.ctx, 0u);
                if (__builtin_expect(nb != 4u, 0)) flag_pair<Lay<NB>::LW>(dt.base_s, dt.ctx, 1u);
            }
            ib += 4 * NS;
        }
    }
    for (int i = ib + h; i < i1; i += NS) {                   // ragged tail (and every ion when the clamp is needed)
        const uint32_t a = ions_s + (uint32_t)(i >> 2) * 48u + (uint32_t)(i & 3) * 4u;
        float dx, dy, dz;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(dx) : "r"(a));
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(dy) : "r"(a + 16u));
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(dz) : "r"(a + 32u));
        if (bin_one<kClamp, kDetect, BLK>(dx, dy, dz, n.ax, n.ay, n.az, c, k0, 1u)) flag_pair<Lay<NB>::LW>(dt.base_s, dt.ctx, 0u);
        if (bin_one<kClamp, kDetect, BLK>(dx, dy, dz, n.bx, n.by, n.bz, c, k0, 65536u)) flag_pair<Lay<NB>::LW>(dt.base_s, dt.ctx, 1u);
    }
}

// Epilogue of one direction group (a5 tail, a6, a7) by one set of four service warps.  Service warp q reads TMEM
// lane quarter q = M rows 32q..32q+31 = part blk = q of all 32 direction slots (slot from the lane).  Window bins
// are handled in rounds of 4: each thread scales its 4 partial sums by the phase w^{blk k}, keeps the one whose
// index is q and hands the other three to the partner warps of its set through `exch` (a reduce-scatter over blk).
// Output: mode 0 (ordinary group gi) writes the slot's own direction and, in half-grid mode, the opposite direction
// unless the pair was flagged (bit of `mask`); mode 1 (fix-up group) writes only the opposite direction of the listed pair.
struct EpiOut {
    int cls, n;                          // class of signatures served by this histogram, its ROI ion count (normalisation)
    int mode, gi, g0, f, nfix;           // g0 = first group of the sub-range, f = fix-up group, nfix = listed pairs
    uint32_t *flag;                      // mode 0, half-grid: flag word of this group (read, then reset)
    const uint16_t *fix;
    int *ovf;                            // set to 1 when a slot's DC sum is not N_c: a counter left the exact fp16 range
};
// (Q = the warp's TMEM lane quarter as a compile-time constant: which of the four partial sums of a round stays in the warp and
// which three go to the partners is then fixed in the code instead of being selected at run time)
template <bool kHalf, int NB, bool kMulti, int Q>
__device__ __forceinline__ void epilogue_group(const MmaParams &p, uint32_t acc, const EpiOut &eo, int64_t m, const float2 *phase,
                                            float2 *exch_all, float2 *cand_all, int set, int lane)
{
    constexpr int q = Q;
    const int mode = kHalf ? eo.mode : 0;
    const uint32_t mask = (kHalf && mode == 0) ? *eo.flag : 0u;         // complete: every binning warp has arrived
    const uint32_t acc0 = acc + ((uint32_t)(q * 32) << 16);
    float2 *exch = exch_all + set * (kEpiRound * 4 * 32), *cand = cand_all + set * (4 * 32);
    // one running maximum per spec of the class (a spec's window is a sub-range of the transformed union window)
    // (kMulti = false: the plan has ONE signature -- the common case keeps the single-maximum code of a one-signature kernel)
    constexpr int NSP = kMulti ? kMaxSpecs : 1;
    const int n_specs = kMulti ? p.ss.n_specs : 1;      // the single-signature kernel never touches p.ss (window = union window)
    float best[NSP];
    int kbest[NSP];
#pragma unroll
    for (int sp = 0; sp < NSP; ++sp) { best[sp] = -1.0f; kbest[sp] = !kMulti ? p.k_lo : (sp < n_specs ? p.ss.k_lo[sp] : 0); }
    const bool one_spec = !kMulti || n_specs == 1;
    float dcsum = 0.f;
#pragma unroll 1
    for (int r0 = 0; r0 < p.W; r0 += kEpiRound) {
        uint32_t v[16];
        tmem_ld16(acc0 + (uint32_t)(4 * r0), v);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        float2 keep = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < kEpiRound; ++j) {
            const int w = r0 + j;
            if (w < p.W) {
                const float re = __uint_as_float(v[4 * j]) + __uint_as_float(v[4 * j + 2]) * (1.0f / 2048.0f);
                const float im = -(__uint_as_float(v[4 * j + 1]) + __uint_as_float(v[4 * j + 3]) * (1.0f / 2048.0f));
                const float2 f = phase[(NB == 4 ? q : 2 * q + (lane >> 4)) * p.W + w];
                float2 P = make_float2(f.x * re - f.y * im, f.x * im + f.y * re);
                if (NB == 8) {                           // lanes l and l + 16 hold parts blk = 2q and 2q + 1 of slot l
                    P.x += __shfl_xor_sync(0xffffffffu, P.x, 16);
                    P.y += __shfl_xor_sync(0xffffffffu, P.y, 16);
                }
                if (j == q) keep = P;
                else exch[(j * 4 + q) * 32 + lane] = P;
            }
        }
        if (p.dc_col >= 0 && r0 == 0) {
            // DC check: the sum of this part's counters as the tensor core read them travels in the exchange slot (j = q) that
            // the reduce-scatter never uses; warp q = 0 adds the parts behind the barrier
            float dcv = __uint_as_float(tmem_ld1(acc0 + (uint32_t)p.dc_col));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (NB == 8) dcv += __shfl_xor_sync(0xffffffffu, dcv, 16);
            exch[(q * 4 + q) * 32 + lane].x = dcv;
        }
        if (set == 0) asm volatile("bar.sync 3, 128;" ::: "memory"); else asm volatile("bar.sync 4, 128;" ::: "memory");
        if (p.dc_col >= 0 && r0 == 0 && q == 0)
            dcsum = (exch[0 * 32 + lane].x + exch[5 * 32 + lane].x) + (exch[10 * 32 + lane].x + exch[15 * 32 + lane].x);
        const int w = r0 + q;
        if (w < p.W) {
            float xr = keep.x, xi = keep.y;
#pragma unroll
            for (int o = 1; o < 4; ++o) {
                const float2 e = exch[(q * 4 + ((q + o) & 3)) * 32 + lane];
                xr += e.x; xi += e.y;
            }
            const float pw = xr * xr + xi * xi;
            const int k = p.k_lo + w;
            if (one_spec) {
                if (pw > best[0]) { best[0] = pw; kbest[0] = k; }        // ascending w: lowest k kept on ties
            } else {
#pragma unroll
                for (int sp = 0; sp < NSP; ++sp)
                    if (kMulti && sp < n_specs && p.ss.cls_of[sp] == eo.cls && k >= p.ss.k_lo[sp] && k <= p.ss.k_hi[sp] && pw > best[sp]) {
                        best[sp] = pw; kbest[sp] = k;
                    }
            }
        }
        if (set == 0) asm volatile("bar.sync 3, 128;" ::: "memory"); else asm volatile("bar.sync 4, 128;" ::: "memory");
    }
    if (kHalf && mode == 0 && q == 0 && lane == 0) *eo.flag = 0u;     // every thread of the set has read it (barriers above)
    bool dc_pending = p.dc_col >= 0;
#pragma unroll 1
    for (int sp = 0; sp < n_specs; ++sp) {
        if (kMulti && p.ss.cls_of[sp] != eo.cls) continue;
        float bsel = best[0];
        int ksel = kbest[0];
#pragma unroll
        for (int j = 1; j < NSP; ++j)
            if (j == sp) { bsel = best[j]; ksel = kbest[j]; }
        cand[q * 32 + lane] = make_float2(bsel, __int_as_float(ksel));
        if (set == 0) asm volatile("bar.sync 3, 128;" ::: "memory"); else asm volatile("bar.sync 4, 128;" ::: "memory");
        if (q == 0 && lane < Lay<NB>::G) {                   // (NB = 8: lanes 16..31 carry copies of lanes 0..15)
            constexpr int G = Lay<NB>::G;
            if (dc_pending) {
                // all parts of the slot: 2^-24 * (sum of the counters as fp16 numbers), exact in fp32.  It equals N_c unless
                // some counter went beyond 2048, where the u16 bit pattern stops being the fp16 number of the same value
                const float dc = dcsum;
                const int slot0 = (lane & 1) * (G / 2) + ((lane >> 3) << 2) + ((lane & 7) >> 1);
                const bool live = mode == 0 ? p.perm[eo.gi * G + slot0] >= 0 : eo.f * G + slot0 < eo.nfix;
                if (live && dc * 16777216.0f != (float)eo.n) *eo.ovf = 1;
            }
            float bb = -1.0f;
            int kb = kMulti ? p.ss.k_lo[sp] : p.k_lo;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const float2 c2 = cand[s * 32 + lane];
                const int ck = __float_as_int(c2.y);
                if (c2.x > bb || (c2.x == bb && ck < kb)) { bb = c2.x; kb = ck; }
            }
            // M row (within a part) = chunk * 8 + word * 2 + half  ->  slot = half * G/2 + chunk * 4 + word
            const int slot = (lane & 1) * (G / 2) + ((lane >> 3) << 2) + ((lane & 7) >> 1);
            float amp = 16777216.0f * sqrtf(fmaxf(bb, 0.0f));
            if (kMulti ? p.ss.norm[sp] : p.norm0) amp = eo.n ? __fdiv_rn(amp, (float)eo.n) : 0.0f;   // normalised intensity A / N_c (L424)
            const float2 res = make_float2(amp, (float)kb);
            float2 *out = p.sig + (kMulti ? (size_t)sp * (size_t)p.M * p.D : (size_t)0) + (size_t)m * p.D;
            if (mode == 0) {
                const int d = p.perm[eo.gi * G + slot];
                if (d >= 0) out[d] = res;
                if (kHalf && !((mask >> slot) & 1u)) {               // the mirrored histogram has the same amplitude spectrum
                    const int d2 = p.perm_mirror[eo.gi * G + slot];
                    if (d2 >= 0) out[d2] = res;
                }
            } else {
                const int e = eo.f * G + slot;
                if (e < eo.nfix) {
                    const int d2 = p.perm_mirror[eo.g0 * G + (int)eo.fix[e]];
                    if (d2 >= 0) out[d2] = res;
                }
            }
        }
        dc_pending = false;
        if (!one_spec) {                                     // cand is reused by the next spec of the class
            if (set == 0) asm volatile("bar.sync 3, 128;" ::: "memory"); else asm volatile("bar.sync 4, 128;" ::: "memory");
        }
    }
    // the set's cand is rewritten only after the barriers of the rounds of its next epilogue
}

// Test hook behind apx_debug_histograms: the MMA warp copies the group's histogram out of the shared-memory buffer the
// binning warps have just filled (and the tensor core is about to read) into uint32[nd][B], un-interleaving the u16
// halves: (bin b, slot) lives in half (slot / LW) of word (slot % LW) at byte (w/4)*SBO + (w%4)*4 + 16*hi3 + BLK*low.
// Pass 0 of a group stores, later passes of a ROI with more than 2048 ions add.  Half-grid mode: the mirrored direction
// gets the histogram reversed (b -> B-1-b) unless the pair is flagged; flagged pairs are stored by their fix-up group.
struct ExportArgs {                      // by value: taking the address of the kernel's parameter block would force a local copy
    uint32_t *hist_out;
    const int *perm, *perm_mirror;
    int hist_d0, hist_nd, B, nl;
};
template <int NB, bool kHalf>
__device__ __noinline__ void export_hist(const ExportArgs p, const unsigned char *hist, int mode, int gi, int g0, int f, int nfix,
                                         const uint16_t *fix, uint32_t mask, int pass, int lane)
{
    constexpr int G = Lay<NB>::G, LW = Lay<NB>::LW, SBO = Lay<NB>::SBO, BLK = Lay<NB>::BLK;
    const int B = p.B, lowmask = (B >> 3) - 1;
    for (int idx = lane; idx < B * G; idx += 32) {
        const int b = idx / G, slot = idx % G, w = slot % LW, hf = slot / LW;
        const int hi3 = b >> p.nl, low = b & lowmask;
        const uint32_t v = *reinterpret_cast<const uint16_t *>(hist + (w >> 2) * SBO + (w & 3) * 4 + 16 * hi3 + BLK * low + 2 * hf);
        int d = -1, d2 = -1;
        if (mode == 0) {
            d = p.perm[gi * G + slot];
            if (kHalf && !((mask >> slot) & 1u)) d2 = p.perm_mirror[gi * G + slot];
        } else {
            const int e = f * G + slot;
            if (e < nfix) d = p.perm_mirror[g0 * G + (int)fix[e]];      // binned as the direction opposite to the listed slot's
        }
        if (d >= p.hist_d0 && d < p.hist_d0 + p.hist_nd) {
            uint32_t *o = p.hist_out + (size_t)(d - p.hist_d0) * B + b;
            *o = pass ? *o + v : v;
        }
        if (d2 >= p.hist_d0 && d2 < p.hist_d0 + p.hist_nd) {
            uint32_t *o = p.hist_out + (size_t)(d2 - p.hist_d0) * B + (B - 1 - b);
            *o = pass ? *o + v : v;
        }
    }
    __syncwarp();
}

// A sequence of direction groups for run_pipeline.  mode 0: the ordinary groups [g0, g0 + ngrp) of the plan's slot
// order.  mode 1: fix-up groups of the half-grid mode, built from the list of flagged pairs of the sub-range that
// starts at group g0 (slot s of fix-up group f = list entry 32 f + s, binned as the direction OPPOSITE to the
// slot's).  grp_base = groups this CTA has run before the sequence: buffer / accumulator / mbarrier parities
// continue across sequences.
struct Seq {
    int mode, g0, ngrp, grp_base, nfix;
};
struct PipeShared {
    uint64_t *full, *done, *doneq, *free_, *epi, *tfree;    // doneq[buf * 3 + q]: first three quarters of a buffer's MMAs complete
    FixShared *fs;
    uint32_t *flag;
    int *n, *nfix;
    uint16_t *fix;
    int *ovf;                                               // 1: this CTA's material point goes to the deferred list
};

// The warp-specialised pipeline of one (material point, chunk).  kBig: the ROI's ions have spilled into the second
// histogram buffer, so only buffer 0 is used and bin -> transform -> clear are serial per item.
template <int KS, int NB, bool kBig, bool kHalf, bool kMulti, int kRole>
__device__ __forceinline__ void run_pipeline(const MmaParams &p, const MmaSmem &L, unsigned char *smem, uint32_t tmem, int n_ions,
                                             const Seq &sq, int64_t m, const float *ions, const float2 *phase,
                                             float2 *exch, float2 *cand, const PipeShared &ps, int cls)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);      // provably warp-uniform: ion addresses live in uniform registers
    // Pipeline over items = (direction group, ion pass); item number itg (counted from the start of the CTA) uses
    // histogram buffer itg & 1, group number gq the TMEM accumulator gq & 1:
    //   binning warps 0..15 : wait free(buf) -> project-and-bin the item -> arrive full(buf)
    //   MMA warp 16         : wait full(buf) [, tfree(acc)] -> K/16 tcgen05.mma -> commit to done(buf) [, epi(acc)]
    //   clear warp 17       : wait done(buf) -> clear the buffer -> free(buf)
    //   service warps 18..25: set s = gq & 1: wait epi(acc) -> epilogue from TMEM -> arrive tfree(acc), acc = gq & (nacc - 1)
    // A ROI with more than `cap` ions has spilled into the second histogram buffer: it runs with buffer 0 only
    // (bin -> transform -> clear serial per item); `use` counts the uses of a buffer.
    const int n = n_ions;
    const int npass = n > p.pass_ions ? (n + p.pass_ions - 1) / p.pass_ions : 1;     // (fp16 counters are exact up to 2048)
    const int nitems = sq.ngrp * npass;
    const int mode = kHalf ? sq.mode : 0;
    const int it_base = sq.grp_base * npass;
#ifdef APX_TRACE
    int trace_n = sq.grp_base == 0 && sq.mode == 0 && cls == 0 ? 0 : (1 << 30);      // the CTA's first sequence only
#endif
    if (kRole == 0) {                                            // (the binning warps; every other warp runs the kRole = 1 copy)
        BinConst c;
        c.half_b = (float)(p.B / 2); c.magic_a = magic_for(p.B); c.magic_b = 12582912.0f + 4.0f;
        c.scl = __int_as_float((127 - p.nl) << 23);                       // 2^-nl
        constexpr int G = Lay<NB>::G, LW = Lay<NB>::LW;
        c.kz = 16u - (uint32_t)Lay<NB>::BLK * (1u << p.nl);
        const int l = lane & (LW - 1), h = lane / LW;
        const uint32_t k0base = smem_u32(smem + L.hist0) + (uint32_t)(l >> 2) * Lay<NB>::SBO + (uint32_t)(l & 3) * 4u
                                - 0x4B400000u * (uint32_t)Lay<NB>::BLK - 0x4B400000u * c.kz;
        const uint32_t ions_s = smem_u32(ions);
        const bool detect = kHalf && mode == 0;
        for (int it = 0, gl = 0, pass = 0; it < nitems; ++it) {
            const int itg = it_base + it, buf = kBig ? 0 : (itg & 1), use = kBig ? itg : (itg >> 1);
            APX_TRACE_EVENT(p, 10, sq.grp_base + gl);                                // loop top
            LaneDirs n;
            if (mode == 0) {
                const float *da = p.dirs_sorted + (size_t)((sq.g0 + gl) * G + l) * 3;
                n.ax = da[0]; n.ay = da[1]; n.az = da[2]; n.bx = da[3 * LW]; n.by = da[3 * LW + 1]; n.bz = da[3 * LW + 2];
            } else {                                                     // the opposite of a flagged pair's direction
                const int ea = gl * G + l, eb = ea + LW;
                const float *da = p.dirs_sorted + (ea < sq.nfix ? (size_t)(sq.g0 * G + (int)ps.fix[ea]) * 3 : 0);
                const float *db = p.dirs_sorted + (eb < sq.nfix ? (size_t)(sq.g0 * G + (int)ps.fix[eb]) * 3 : 0);
                n.ax = -da[0]; n.ay = -da[1]; n.az = -da[2]; n.bx = -db[0]; n.by = -db[1]; n.bz = -db[2];
            }
            APX_TRACE_EVENT(p, 0, sq.grp_base + gl);                                 // binning warp ready for the item
            if (kBig) {
                // single-buffered: the shared-memory pipe is idle while the tensor core transforms the buffer, so the 16
                // binning warps clear it themselves as soon as it has been read (a few STS.128 per thread)
                if (use >= 1) {
                    mbar_wait(&ps.done[0], (uint32_t)((use - 1) & 1));
                    uint4 *hb = reinterpret_cast<uint4 *>(smem + L.hist0);
                    for (int i = tid; i < (int)(L.hist_bytes / 16); i += kBinWarps * 32) hb[i] = make_uint4(0, 0, 0, 0);
                    asm volatile("bar.sync 5, %0;" ::"n"(kBinWarps * 32) : "memory");
                }
            } else if (use >= 1) {
                mbar_wait_lean(&ps.free_[buf], (uint32_t)((use - 1) & 1));             // cleared after its previous use
            }
            APX_TRACE_EVENT(p, 1, sq.grp_base + gl);                                 // bin start (buffer free)
            const int a0 = pass * p.pass_ions, a1 = min(n_ions, a0 + p.pass_ions);
            int i0, i1;
            if (p.unit_split) {                                                      // whole blocks of 4 * NS ions per warp: no ragged tails
                constexpr int U = 4 * Lay<NB>::NS;
                const int nu = (a1 - a0 + U - 1) / U;
                i0 = a0 + U * ((warp * nu) / kBinWarps); i1 = min(a1, a0 + U * (((warp + 1) * nu) / kBinWarps));
            } else {
                const int nq = (a1 - a0 + 3) >> 2;                                   // quads of this pass, split evenly
                i0 = a0 + 4 * ((warp * nq) / kBinWarps); i1 = min(a1, a0 + 4 * (((warp + 1) * nq) / kBinWarps));
            }
            uint32_t k0 = k0base + (uint32_t)buf * (L.hist1 - L.hist0);
            // opaque to the compiler: it would otherwise re-derive k0 and kz from the thread id and the shared-memory base
            // (S2R, shifts, multiplies: ~20 of 146 instructions) in every iteration of the binning loop
            asm volatile("mov.b32 %0, %0;" : "+r"(k0));
            asm volatile("mov.b32 %0, %0;" : "+r"(c.kz));
            Detect dt;
            dt.base_s = dt.ctx = 0u;
            if (detect) {
                dt.base_s = smem_u32(ps.fs);
                dt.ctx = (uint32_t)((sq.grp_base + gl) & (kFlagSlots - 1)) | ((uint32_t)l << 4) | ((uint32_t)(gl * G) << 16);
                asm volatile("mov.b32 %0, %0;" : "+r"(dt.base_s));
                asm volatile("mov.b32 %0, %0;" : "+r"(dt.ctx));
                bin_ions<false, true, NB>(ions_s, i0, i1, n, c, k0, h, dt);
            } else if (p.clamp) {
                bin_ions<true, false, NB>(ions_s, i0, i1, n, c, k0, h, dt);
            } else {
                bin_ions<false, false, NB>(ions_s, i0, i1, n, c, k0, h, dt);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // histogram writes -> async proxy
            __syncwarp();
            APX_TRACE_EVENT(p, 2, sq.grp_base + gl);                                 // bin end
            if (lane == 0) mbar_arrive(&ps.full[buf]);
            APX_TRACE_EVENT(p, 9, sq.grp_base + gl);                                 // arrived
            if (++pass == npass) { pass = 0; ++gl; }
        }
    } else if (kRole != 0 && warp == kMmaWarp) {
        // ---- MMA warp: descriptors advance by adding to the 14-bit start-address field ---------------
        const uint32_t idesc = (1u << 4) | (1u << 15) | ((uint32_t)(p.N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        const uint32_t tb = smem_u32(smem + L.table), hb = smem_u32(smem + L.hist0);
        const uint32_t a_hi = (uint32_t)(Lay<NB>::SBO >> 4) | (1u << 14);                        // SBO, version 1, INTERLEAVE
        const uint32_t a_lo0 = ((hb >> 4) & 0x3FFFu) | ((uint32_t)(Lay<NB>::LBO >> 4) << 16);      // LBO
        const uint32_t b_hi = (uint32_t)(1024 >> 4) | (1u << 14) | (2u << 29);                     // SBO, version 1, SWIZZLE_128B
        const uint32_t b_lo0 = ((tb >> 4) & 0x3FFFu) | (1u << 16);
        const uint32_t kblk_step = (uint32_t)(p.N * 128) >> 4;
        for (int it = 0, gl = 0, pass = 0; it < nitems; ++it) {
            const int itg = it_base + it, buf = kBig ? 0 : (itg & 1), use = kBig ? itg : (itg >> 1);
            const int gq = sq.grp_base + gl;
            mbar_wait<100>(&ps.full[buf], (uint32_t)(use & 1));
            APX_TRACE_EVENT(p, 3, gq);                                                // MMA warp: buffer full
            if (pass == 0 && gq >= p.nacc) mbar_wait(&ps.tfree[gq & (p.nacc - 1)], (uint32_t)(((gq >> p.nacc_log2) - 1) & 1));
            APX_TRACE_EVENT(p, 4, gq);                                                // accumulator free, MMAs issued next
            asm volatile("tcgen05.fence::after_thread_sync;");
            if (p.hist_out && cls == 0)                          // test hook (first class): the buffer is complete
                export_hist<NB, kHalf>(ExportArgs{p.hist_out, p.perm, p.perm_mirror, p.hist_d0, p.hist_nd, p.B, p.nl},
                                       smem + (buf ? L.hist1 : L.hist0), mode, sq.g0 + gl, sq.g0, gl, sq.nfix, ps.fix,
                                       (kHalf && mode == 0) ? ps.flag[gq & (kFlagSlots - 1)] : 0u, pass, lane);
            const uint32_t acc = tmem + (uint32_t)((gq & (p.nacc - 1)) * p.N);
            if (lane == 0) {
                const uint32_t a_lo = a_lo0 + (uint32_t)buf * ((L.hist1 - L.hist0) >> 4);
#pragma unroll
                for (int ks = 0; ks < KS; ++ks) {
                    const uint64_t ad = ((uint64_t)a_hi << 32) | (a_lo + (uint32_t)ks * ((2 * Lay<NB>::LBO) >> 4));
                    const uint64_t bd = ((uint64_t)b_hi << 32) | (b_lo0 + (uint32_t)(ks >> 2) * kblk_step + (uint32_t)(ks & 3) * 2u);
                    if (ks == 0) mma_f16_ss(acc, ad, bd, idesc, pass > 0 ? 1u : 0u);
                    else mma_f16_acc(acc, ad, bd, idesc);
                    // k-steps 4q..4q+3 read the q-th quarter of the buffer (contiguous bytes): a commit per quarter lets the
                    // clear warp zero it while the remaining MMAs still run
                    if (!kBig && KS >= 4 && (ks + 1) % (KS / 4) == 0 && ks + 1 < KS)
                        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                     ::"r"(smem_u32(&ps.doneq[buf * 3 + (ks + 1) / (KS / 4) - 1])) : "memory");
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                             ::"r"(smem_u32(&ps.done[buf])) : "memory");
                if (pass == npass - 1)                                           // the group's accumulator is complete
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                 ::"r"(smem_u32(&ps.epi[gq & (p.nacc - 1)])) : "memory");
            }
            __syncwarp();
            if (++pass == npass) { pass = 0; ++gl; }
        }
    } else if (kRole != 0 && warp == kClrWarp) {
        // ---- clear warp: once the tensor core has read a buffer, clear it with bulk copies of zeros (TMA engine, no
        //      LSU work); free(buf) completes when all bytes have landed
        for (int it = 0; it < (kBig ? 0 : nitems); ++it) {           // (single-buffered: the binning warps clear)
            const int itg = it_base + it, buf = kBig ? 0 : (itg & 1), use = kBig ? itg : (itg >> 1);
            const uint32_t piece = L.hist_bytes / 4;
            if (n >= kStsClearBelow && lane == 0)
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&ps.free_[buf])), "r"(L.hist_bytes) : "memory");
#pragma unroll 1
            for (int c4 = 0; c4 < 4; ++c4) {                     // quarter by quarter, as the tensor core releases them
                mbar_wait<100>(c4 < 3 ? &ps.doneq[buf * 3 + c4] : &ps.done[buf], (uint32_t)(use & 1));
                if (c4 == 3) APX_TRACE_EVENT(p, 5, it_base + it);                     // clear warp: all MMAs of the buffer done
                if (n < kStsClearBelow) {
                    // few ions: the LSU pipe has room, clear with plain stores and spare the L2 the zero traffic
                    uint4 *hp = reinterpret_cast<uint4 *>(smem + (buf ? L.hist1 : L.hist0) + c4 * piece);
                    for (int i = lane; i < (int)(piece / 16); i += 32) hp[i] = make_uint4(0, 0, 0, 0);
                } else if (lane == 0) {
                    const uint32_t dst = smem_u32(smem + (buf ? L.hist1 : L.hist0)), bar = smem_u32(&ps.free_[buf]);
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(dst + c4 * piece), "l"((const char *)p.zeros + c4 * piece), "r"(piece), "r"(bar) : "memory");
                }
            }
            if (n < kStsClearBelow) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&ps.free_[buf]);
            }
            __syncwarp();
        }
    } else if (kRole != 0) {
        // ---- service warps: set s runs the epilogue of the groups with (group number & 1) == s ----------
        const int q = warp & 3, set = (warp - kSvcWarp0) >> 2;
        for (int gl = (set ^ sq.grp_base) & 1; gl < sq.ngrp; gl += 2) {
            const int gq = sq.grp_base + gl;
            mbar_wait_lean<200>(&ps.epi[gq & (p.nacc - 1)], (uint32_t)((gq >> p.nacc_log2) & 1));
            APX_TRACE_EVENT(p, 7, gq);                                                // epilogue start
            asm volatile("tcgen05.fence::after_thread_sync;");
            EpiOut eo;
            eo.cls = cls; eo.n = n;
            eo.mode = mode; eo.gi = sq.g0 + gl; eo.g0 = sq.g0; eo.f = gl; eo.nfix = sq.nfix;
            eo.flag = kHalf ? &ps.flag[gq & (kFlagSlots - 1)] : nullptr; eo.fix = ps.fix; eo.ovf = ps.ovf;
            const uint32_t acc_g = tmem + (uint32_t)((gq & (p.nacc - 1)) * p.N);
            switch (q) {                                                            // (warp-uniform)
                case 0: epilogue_group<kHalf, NB, kMulti, 0>(p, acc_g, eo, m, phase, exch, cand, set, lane); break;
                case 1: epilogue_group<kHalf, NB, kMulti, 1>(p, acc_g, eo, m, phase, exch, cand, set, lane); break;
                case 2: epilogue_group<kHalf, NB, kMulti, 2>(p, acc_g, eo, m, phase, exch, cand, set, lane); break;
                default: epilogue_group<kHalf, NB, kMulti, 3>(p, acc_g, eo, m, phase, exch, cand, set, lane); break;
            }
            asm volatile("tcgen05.fence::before_thread_sync;");
            __syncwarp();
            APX_TRACE_EVENT(p, 8, gq);                                                // epilogue end
            if (lane == 0) mbar_arrive(&ps.tfree[gq & (p.nacc - 1)]);
        }
    }
}

// one sequence, in the double-buffered pipeline or -- the ROI's ions have spilled into the second buffer, or B = 2048 -- the
// single-buffered one
template <int KS, int NB, bool kHalf, bool kMulti, int kRole>
__device__ __forceinline__ void run_seq(const MmaParams &p, const MmaSmem &L, unsigned char *smem, uint32_t tmem, int n, const Seq &sq,
                                        int64_t m, const float *ions, const float2 *phase, float2 *exch, float2 *cand,
                                        const PipeShared &ps, int cls)
{
    if (NB == 8 || n > p.cap) run_pipeline<KS, NB, true, kHalf, kMulti, kRole>(p, L, smem, tmem, n, sq, m, ions, phase, exch, cand, ps, cls);
    else run_pipeline<KS, NB, false, kHalf, kMulti, kRole>(p, L, smem, tmem, n, sq, m, ions, phase, exch, cand, ps, cls);
}

// (Re-)initialise the pipeline's barriers and counters; one thread.  again: a new class of signatures restarts the phase counts.
__device__ __forceinline__ void init_barriers(const PipeShared &ps, bool again)
{
    auto reinit = [&](uint64_t *b, uint32_t cnt) {
        if (again) asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
        mbar_init(b, cnt);
    };
    for (int i = 0; i < 2; ++i) { reinit(&ps.full[i], kBinWarps); reinit(&ps.done[i], 1); reinit(&ps.free_[i], 1); }
    for (int i = 0; i < 6; ++i) reinit(&ps.doneq[i], 1);
    for (int i = 0; i < 4; ++i) { reinit(&ps.epi[i], 1); reinit(&ps.tfree[i], 4); }
    asm volatile("fence.mbarrier_init.release.cluster;");
    *ps.n = 0; *ps.nfix = 0; *ps.ovf = 0;
    for (int i = 0; i < kFlagSlots; ++i) ps.flag[i] = 0u;
}

// A fix-list overflow or a failed DC check (a counter beyond 2048 in a single-pass ROI) sends the material point to the FFT
// kernel: at most one entry per CTA and class.  Thread 0, behind a CTA barrier that follows the last epilogue of the class.
__device__ __forceinline__ void flush_overflow(const MmaParams &p, const PipeShared &ps, int64_t m)
{
    if (*ps.ovf) {
        p.deferred[1 + atomicAdd(&p.deferred[0], 1u)] = (uint32_t)m;
        *ps.ovf = 0;
    }
}

// Work of one CTA = (material point m, chunk of direction groups [g_begin, g_end)) after the setup: one pass per class of
// signatures (specs with the same type mask): gather, then the group pipeline.  Compiled twice: kRole 0 is the copy the
// 16 binning warps run (they also gather), kRole 1 the copy of the MMA, clear and service warps.  Both copies execute the
// same sequence of CTA-wide barriers.  The split keeps the other roles' code (and their live registers) out of the binning
// warps' copy, so that the constants of the binning loop stay in registers.
struct CtaWork {
    int chunk, g_begin, g_end;
    int64_t m;
    float cx, cy, cz;
};
template <int KS, int NB, bool kHalf, bool kMulti, int kRole>
__device__ __forceinline__ void cta_body(const MmaParams &p, const MmaSmem &L, unsigned char *smem, const PipeShared &ps,
                                         const uint32_t *s_tmem, const CtaWork &w, uint32_t &tmem)
{
    const int tid = threadIdx.x, warp = tid >> 5;
    const int chunk = w.chunk, g_begin = w.g_begin, g_end = w.g_end;
    const int64_t m = w.m;
    float *ions = reinterpret_cast<float *>(smem + L.ions);
    float2 *exch = reinterpret_cast<float2 *>(smem + L.exch);
    float2 *cand = reinterpret_cast<float2 *>(smem + L.cand);
    float2 *phase = reinterpret_cast<float2 *>(smem + L.phase);
    const int n_classes = kMulti ? p.ss.n_classes : 1;
    for (int cls = 0; cls < n_classes; ++cls) {
        if (cls > 0) {
            __syncthreads();                               // the previous class has drained (epilogues done, clears landed)
            if (tid == 0) {
                flush_overflow(p, ps, m);
                init_barriers(ps, true);
            }
        }
        {
            uint4 *h0 = reinterpret_cast<uint4 *>(smem + L.hist0), *h1 = reinterpret_cast<uint4 *>(smem + L.hist1);
            for (int i = tid; i < (int)(L.hist_bytes / 16); i += kMmaThreads) {
                h0[i] = make_uint4(0, 0, 0, 0);
                if (NB == 4) h1[i] = make_uint4(0, 0, 0, 0);
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;");
        tmem = *s_tmem;
        if (kRole == 0) {                                  // (the binning warps gather)
            const GridParams g = *p.grid;
            if (g.n_accepted) {
                const RoiCells rc = roi_cells(g, w.cx, w.cy, w.cz, p.R);
                gather_roi3<kMulti>(p, g, rc, w.cx, w.cy, w.cz, ions, ps.n, cls, kBinWarps);
            }
        }
        __syncthreads();
        const int n = *ps.n;
        if (chunk == 0 && tid == 0 && p.counts) {
            if (!kMulti) p.counts[m] = (uint32_t)n;
            else
                for (int sp = 0; sp < p.ss.n_specs; ++sp)
                    if (p.ss.cls_of[sp] == cls) p.counts[(size_t)sp * p.M + m] = (uint32_t)n;
        }

        if (n == 0 && !p.hist_out) {
            // empty ROI (e.g. a material point in the other phase of a filtered run): every histogram is zero, so every
            // amplitude is 0 and the arg-max keeps the lowest bin of the window -- written without running the pipeline
            constexpr int G = Lay<NB>::G;
            for (int sl = g_begin * G + tid; sl < g_end * G; sl += kMmaThreads) {
                const int d = p.perm[sl], d2 = kHalf ? p.perm_mirror[sl] : -1;
                const int n_specs = kMulti ? p.ss.n_specs : 1;
                for (int sp = 0; sp < n_specs; ++sp) {
                    if (kMulti && p.ss.cls_of[sp] != cls) continue;
                    float2 *out = p.sig + (kMulti ? (size_t)sp * (size_t)p.M * p.D : (size_t)0) + (size_t)m * p.D;
                    const float2 res = make_float2(0.0f, (float)(kMulti ? p.ss.k_lo[sp] : p.k_lo));
                    if (d >= 0) out[d] = res;
                    if (d2 >= 0) out[d2] = res;
                }
            }
            continue;
        }
        int grp_total = 0;                                     // groups run by this CTA for this class (ordinary + fix-up)
        if (n > p.cap_big) {
            // too many ions even for ion buffer + second histogram buffer: leave this material point to the FFT kernel
            if (chunk == 0 && tid == 0) p.deferred[1 + atomicAdd(&p.deferred[0], 1u)] = (uint32_t)m;
        } else {
            // half-grid mode: sub-ranges of kSubGroups groups, each followed by the fix-up groups of its flagged pairs
            const int sub = kHalf ? kSubGroups : (g_end - g_begin);
            bool overflow = false;
            for (int sg = g_begin; sg < g_end; sg += sub) {
                Seq sq;
                sq.mode = 0; sq.g0 = sg; sq.ngrp = min(sub, g_end - sg); sq.grp_base = grp_total; sq.nfix = 0;
                run_seq<KS, NB, kHalf, kMulti, kRole>(p, L, smem, tmem, n, sq, m, ions, phase, exch, cand, ps, cls);
                grp_total += sq.ngrp;
                if (kHalf) {
                    __syncthreads();                           // every epilogue of the sub-range is done, the list is complete
                    const int nf = *ps.nfix;
                    __syncthreads();
                    if (tid == 0) *ps.nfix = 0;
                    if (nf > kFixCap) overflow = true;         // pathological input: the FFT kernel redoes this material point
                    sq.mode = 1; sq.nfix = min(nf, kFixCap); sq.ngrp = (sq.nfix + Lay<NB>::G - 1) / Lay<NB>::G; sq.grp_base = grp_total;
                    if (sq.ngrp) run_seq<KS, NB, kHalf, kMulti, kRole>(p, L, smem, tmem, n, sq, m, ions, phase, exch, cand, ps, cls);
                    grp_total += sq.ngrp;
                    __syncthreads();                           // the list is consumed before the next sub-range appends
                }
            }
            if (overflow && tid == 0) *ps.ovf = 1;
            // the bulk copies that clear the buffers after their last use must land before the CTA gives up its shared memory
            // (or re-initialises the barriers for the next class)
            if (kRole != 0 && warp == kClrWarp && grp_total > 0) {
                const int npass = n > p.pass_ions ? (n + p.pass_ions - 1) / p.pass_ions : 1, items = grp_total * npass;
                if (NB == 8 || n > p.cap) {
                    // single-buffered: cleared with plain stores by the binning warps, nothing in flight
                } else {
                    const int u0 = (items + 1) >> 1, u1 = items >> 1;
                    if (u0) mbar_wait(&ps.free_[0], (uint32_t)((u0 - 1) & 1));
                    if (u1) mbar_wait(&ps.free_[1], (uint32_t)((u1 - 1) & 1));
                }
            }
        }
    }
}

// KS = K/16 k-steps per group, NB = bin parts (layout), kHalf = half-grid mode, kMulti = several signatures per plan
template <int KS, int NB, bool kHalf, bool kMulti>
__global__ void __launch_bounds__(kMmaThreads, 1) k_signature_mma(const __grid_constant__ MmaParams p)
{
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 1024-byte aligned, still shared-space
    const MmaSmem L = mma_smem_layout(p.B, p.N, p.W, p.cap);
    // per histogram buffer: full (binned), done (transformed), free (cleared); per accumulator: tfree (read out)
    __shared__ uint64_t s_full[2], s_done[2], s_doneq[6], s_free[2], s_epi[4], s_tfree[4];      // per histogram buffer / per accumulator
    __shared__ uint32_t s_tmem;
    __shared__ int s_n, s_ovf;
    __shared__ FixShared s_fs;

    const int tid = threadIdx.x, warp = tid >> 5;
    // CTAs are ordered chunk-major; with up to 6 chunks per material point the chunks shrink geometrically (weights
    // 2^(nchunks-1-c)), so the last waves of the grid consist of the smallest work items
    CtaWork w;
    w.chunk = blockIdx.x / p.M;
    w.m = blockIdx.x % p.M;
    if (p.nchunks <= 6) {
        const int wtot = (1 << p.nchunks) - 1, wlo = wtot - ((1 << (p.nchunks - w.chunk)) - 1);
        w.g_begin = (int)((int64_t)wlo * p.ngroups / wtot);
        w.g_end = (int)((int64_t)(wlo + (1 << (p.nchunks - 1 - w.chunk))) * p.ngroups / wtot);
    } else {                                                   // few material points: many equal chunks
        w.g_begin = (int)((int64_t)w.chunk * p.ngroups / p.nchunks);
        w.g_end = (int)((int64_t)(w.chunk + 1) * p.ngroups / p.nchunks);
    }
    w.cx = p.centres[3 * w.m]; w.cy = p.centres[3 * w.m + 1]; w.cz = p.centres[3 * w.m + 2];
    constexpr int K = KS * 16;

    // ---- setup: barriers, TMEM, twiddle table ----------------------------------------------------------
    PipeShared ps;
    ps.full = s_full; ps.done = s_done; ps.doneq = s_doneq; ps.free_ = s_free; ps.epi = s_epi; ps.tfree = s_tfree;
    ps.fs = &s_fs; ps.flag = s_fs.flag; ps.n = &s_n; ps.nfix = &s_fs.nfix; ps.fix = s_fs.fix; ps.ovf = &s_ovf;
    if (tid == 0) init_barriers(ps, false);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "r"(p.tmem_cols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    {
        uint4 *t = reinterpret_cast<uint4 *>(smem + L.table);
        float2 *phase = reinterpret_cast<float2 *>(smem + L.phase);
        for (int i = tid; i < K * p.N / 8; i += kMmaThreads) t[i] = p.table[i];
        for (int i = tid; i < NB * p.W; i += kMmaThreads) phase[i] = p.phase[i];
    }
    uint32_t tmem = 0;
    if (warp < kBinWarps) cta_body<KS, NB, kHalf, kMulti, 0>(p, L, smem, ps, &s_tmem, w, tmem);
    else cta_body<KS, NB, kHalf, kMulti, 1>(p, L, smem, ps, &s_tmem, w, tmem);
    // ---- teardown ---------------------------------------------------------------------------------
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (tid == 0) flush_overflow(p, ps, w.m);
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(p.tmem_cols));
}

// ---- host side ------------------------------------------------------------------------------------
static int mma_n_for(int W) { return ((4 * W + 15) / 16) * 16; }
static int mma_cap_for(int B, int N, int W)
{
    const int budget = 232448 - 1280;  // 227 KB opt-in shared memory per CTA on sm_100, minus static shared (barriers, fix list)
    MmaSmem s = mma_smem_layout(B, N, W, 0);
    int cap = ((budget - (int)s.total) / 12) & ~63;
    return cap > 4096 ? 4096 : cap;
}

bool mma_path_supported(const Plan *p)
{
    if (p->B > 2048) return false;                       // B = 4096 stays on the FFT kernel
    const int N = mma_n_for(p->W);
    if (2 * N > 512) return false;                       // two accumulators of N TMEM columns
    return mma_cap_for(p->B, N, p->W) >= 1024;           // room for a useful ion buffer
}

// Direction order of the binning warps.  A group of 32 slots = a compact patch of 16 directions (set A, lanes 0..15)
// followed by the 16 directions nearest to the ANTIPODE of that patch (set B, lanes 16..31).  Within one shared atomic
// the 16 lanes of a half-warp project the ion onto nearly parallel directions, so their bins share the top three bits
// (hi3) and hit 16 different banks; the other half-warp sees x -> -x, hi3 -> 7 - hi3, the other bank parity.
// Construction: fold every direction onto one hemisphere (f = n or -n), split into the unflipped set P and the flipped
// set Q (equal sizes for Fibonacci grids with even D and for antipodally symmetric grids; otherwise balanced by
// moving the surplus), then bisect P and Q in lockstep along the widest axis of the folded coordinates, cutting both
// at the same multiple of 16.  The order only affects bank conflicts, never results.
struct FoldedDir {
    float f[3];
    int idx;
};
static void pair_bisect(std::vector<FoldedDir> &P, std::vector<FoldedDir> &Q, int lo, int hi, int leaf)
{
    const int cnt = hi - lo;
    const int pe = std::min(hi, (int)P.size()), qe = std::min(hi, (int)Q.size());
    auto lex = [](const FoldedDir &a, const FoldedDir &b) {
        return a.f[0] != b.f[0] ? a.f[0] < b.f[0] : (a.f[1] != b.f[1] ? a.f[1] < b.f[1] : a.f[2] < b.f[2]);
    };
    if (cnt <= leaf) {                                   // leaf: same slot order on both sides (exact antipodes line up)
        if (lo < pe) std::sort(P.begin() + lo, P.begin() + pe, lex);
        if (lo < qe) std::sort(Q.begin() + lo, Q.begin() + qe, lex);
        return;
    }
    float mn[3] = {1e30f, 1e30f, 1e30f}, mx[3] = {-1e30f, -1e30f, -1e30f};
    for (int i = lo; i < pe; ++i)
        for (int a = 0; a < 3; ++a) { mn[a] = std::min(mn[a], P[i].f[a]); mx[a] = std::max(mx[a], P[i].f[a]); }
    for (int i = lo; i < qe; ++i)
        for (int a = 0; a < 3; ++a) { mn[a] = std::min(mn[a], Q[i].f[a]); mx[a] = std::max(mx[a], Q[i].f[a]); }
    int ax = 0;
    for (int a = 1; a < 3; ++a)
        if (mx[a] - mn[a] > mx[ax] - mn[ax]) ax = a;
    const int leaves = (cnt + leaf - 1) / leaf;
    const int mid = lo + (leaves / 2) * leaf;
    auto cmp = [&](const FoldedDir &a, const FoldedDir &b) { return a.f[ax] != b.f[ax] ? a.f[ax] < b.f[ax] : lex(a, b); };
    if (mid < pe) std::nth_element(P.begin() + lo, P.begin() + mid, P.begin() + pe, cmp);
    if (mid < qe) std::nth_element(Q.begin() + lo, Q.begin() + mid, Q.begin() + qe, cmp);
    pair_bisect(P, Q, lo, mid, leaf);
    pair_bisect(P, Q, mid, hi, leaf);
}
// v = [D][3]; returns the slot order (original index per slot, -1 = padding), length = multiple of 32
static std::vector<int> pair_order(const std::vector<float> &v, int D, int leaf)
{
    std::vector<FoldedDir> P, Q;
    for (int i = 0; i < D; ++i) {
        const float x = v[3 * (size_t)i], y = v[3 * (size_t)i + 1], z = v[3 * (size_t)i + 2];
        const bool up = z > 0.f || (z == 0.f && (y > 0.f || (y == 0.f && x > 0.f)));
        FoldedDir d;
        d.idx = i;
        for (int a = 0; a < 3; ++a) d.f[a] = up ? v[3 * (size_t)i + a] : -v[3 * (size_t)i + a];
        (up ? P : Q).push_back(d);
    }
    auto move_surplus = [](std::vector<FoldedDir> &big, std::vector<FoldedDir> &small) {
        while (big.size() > small.size() + 1) {          // unbalanced input: the surplus keeps f = -(its folded vector)
            FoldedDir d = big.back();
            big.pop_back();
            for (int a = 0; a < 3; ++a) d.f[a] = -d.f[a];
            small.push_back(d);
        }
    };
    move_surplus(P, Q);
    move_surplus(Q, P);
    const int cnt = (int)std::max(P.size(), Q.size());
    const int leaves = (cnt + leaf - 1) / leaf;
    if (leaves > 0) pair_bisect(P, Q, 0, leaves * leaf, leaf);
    std::vector<int> slots((size_t)leaves * 2 * leaf, -1);
    for (int j = 0; j < leaves; ++j)
        for (int e = 0; e < leaf; ++e) {
            const int i = j * leaf + e;
            if (i < (int)P.size()) slots[(size_t)j * 2 * leaf + e] = P[i].idx;
            if (i < (int)Q.size()) slots[(size_t)j * 2 * leaf + leaf + e] = Q[i].idx;
        }
    return slots;
}

cudaError_t mma_path_prepare(Plan *p)
{
    const int B = p->B, nb = mma_nb_for(B), K = B / nb, W = p->W, N = mma_n_for(W);
    const int G = 128 / nb, leaf = G / 2;               // slots per group, directions per patch
    int nl = 0;
    while ((8 << nl) < B) ++nl;                          // B = 8 * 2^nl
    // twiddle table: K index k = kg*8 + hi3 stands for the bin part hi3*(B/8) + 4*kg
    std::vector<uint16_t> img((size_t)K * N, 0);
    for (int r = 0; r < K; ++r)
        for (int n = 0; n < N; ++n) {
            const int w = n / 4, c = n % 4;
            __half val = __float2half(0.0f);
            if (n == 4 * W) val = __float2half(1.0f);    // spare column (if N > 4 W): "k = 0" twiddle, the DC check of MmaParams::dc_col
            if (w < W) {
                const int64_t binpart = (int64_t)(r & 7) * (B / 8) + nb * (r >> 3);
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
    // recombination phases exp(-2 pi i blk k / B), blk = 0..3
    std::vector<float2> ph((size_t)nb * W);
    for (int pb = 0; pb < nb; ++pb)
        for (int w = 0; w < W; ++w) {
            const int64_t off = pb;
            const double th = 2.0 * M_PI * (double)((off * (p->k_lo + w)) % B) / (double)B;
            ph[(size_t)pb * W + w] = make_float2((float)std::cos(th), (float)-std::sin(th));
        }
    e = cudaMalloc(&p->d_mma_phase, ph.size() * sizeof(float2));
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p->d_mma_phase, ph.data(), ph.size() * sizeof(float2), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;

    const size_t hist_bytes = mma_smem_layout(B, N, W, 0).hist_bytes;
    e = cudaMalloc(&p->d_mma_zero, hist_bytes);
    if (e != cudaSuccess) return e;
    e = cudaMemset(p->d_mma_zero, 0, hist_bytes);
    if (e != cudaSuccess) return e;
    std::vector<float> nps((size_t)3 * p->D);
    e = cudaMemcpy(nps.data(), p->d_dirs_scaled, nps.size() * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return e;
    // Antipodally symmetric grid (every direction has its exact negative in the grid, e.g. the paper's geodesic mesh):
    // half-grid mode bins one member of every pair and writes its result to both directions.
    const int D = p->D;
    std::vector<int> partner((size_t)D, -1);
    bool sym = !p->need_clamp && !(p->desc.flags & APX_FLAG_NO_PAIRING) && D >= 2 && D % 2 == 0;
    if (sym) sym = apx_dirs_antipodes(nps.data(), D, partner.data()) == 1;   // scaling by s keeps n' = -(-n)'
    std::vector<int> perm, mirror;
    std::vector<float> sorted;
    if (sym) {
        // one representative per pair (the member on the upper hemisphere), ordered into compact patches of 16 by the same
        // bisection; a group = patch 2g as it is (set A) and patch 2g+1 NEGATED (set B): the two neighbouring patches then
        // project an ion to x and roughly -x, which puts their histogram rows on different shared-memory banks
        std::vector<FoldedDir> P, Q;
        for (int i = 0; i < D; ++i) {
            const float x = nps[3 * (size_t)i], y = nps[3 * (size_t)i + 1], z = nps[3 * (size_t)i + 2];
            const bool up = z > 0.f || (z == 0.f && (y > 0.f || (y == 0.f && x > 0.f)));
            if (!up) continue;
            FoldedDir d;
            d.idx = i;
            for (int a = 0; a < 3; ++a) d.f[a] = nps[3 * (size_t)i + a];
            P.push_back(d);
        }
        if ((int)P.size() * 2 != D) sym = false;
        else {
            const int npairs = (int)P.size(), leaves = (npairs + leaf - 1) / leaf, ngroups = (leaves + 1) / 2;
            pair_bisect(P, Q, 0, leaves * leaf, leaf);
            perm.assign((size_t)ngroups * G, -1);
            mirror.assign((size_t)ngroups * G, -1);
            sorted.assign((size_t)ngroups * G * 3, 0.0f);
            for (int sl = 0; sl < ngroups * G; ++sl)           // padding: any valid vector
                for (int a = 0; a < 3; ++a) sorted[3 * (size_t)sl + a] = nps[a];
            for (int i = 0; i < npairs; ++i) {
                const int j = i / leaf, e = i % leaf, sl = (j / 2) * G + (j & 1) * leaf + e;
                const int own = (j & 1) ? partner[P[i].idx] : P[i].idx;
                perm[sl] = own; mirror[sl] = partner[own];
                for (int a = 0; a < 3; ++a) sorted[3 * (size_t)sl + a] = nps[3 * (size_t)own + a];
            }
        }
    }
    if (!sym) {
        // paired patch order, padded to a multiple of 32 (padding slots repeat direction 0, perm = -1)
        perm = pair_order(nps, p->D, leaf);
        mirror.clear();
        sorted.assign(perm.size() * 3, 0.0f);
        for (size_t i = 0; i < perm.size(); ++i) {
            const int src = perm[i] >= 0 ? perm[i] : 0;
            for (int a = 0; a < 3; ++a) sorted[3 * i + a] = nps[3 * (size_t)src + a];
        }
    }
    // scheduling knobs: defaults chosen from measurements, overridable from the environment for A/B runs
    p->tune_unit_split = 1; p->tune_nacc = 4;
    if (const char *ev = std::getenv("APX_TUNE_UNITS")) p->tune_unit_split = std::atoi(ev);
    p->tune_dc = 1;
    if (const char *ev = std::getenv("APX_TUNE_DC")) p->tune_dc = std::atoi(ev);
    if (const char *ev = std::getenv("APX_TUNE_NACC")) p->tune_nacc = std::atoi(ev);
    const int Dp = (int)perm.size();
    p->mma_paired = sym ? 1 : 0;
    p->Dp = Dp;
    e = cudaMalloc(&p->d_dirs_sorted, sorted.size() * 4);
    if (e != cudaSuccess) return e;
    e = cudaMalloc(&p->d_dir_perm, perm.size() * 4);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p->d_dirs_sorted, sorted.data(), sorted.size() * 4, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p->d_dir_perm, perm.data(), perm.size() * 4, cudaMemcpyHostToDevice);
    if (e != cudaSuccess || !sym) return e;
    e = cudaMalloc(&p->d_dir_perm_mirror, mirror.size() * 4);
    if (e != cudaSuccess) return e;
    return cudaMemcpy(p->d_dir_perm_mirror, mirror.data(), mirror.size() * 4, cudaMemcpyHostToDevice);
}

// chunks of direction groups per material point: one gather per material point when there are enough of them
static int mma_nchunks_for(const Plan *p, int64_t M)
{
    int nchunks = 1;
    const int slots_per_group = 128 / mma_nb_for(p->B);
    const int ngroups_all = p->Dp / slots_per_group;
    const int64_t want = (int64_t)p->sm_count * 8;
    if (M * nchunks < want) nchunks = (int)((want + M - 1) / M);
    if (nchunks > (ngroups_all + 1) / 2) nchunks = (ngroups_all + 1) / 2;
    if (nchunks < 1) nchunks = 1;
    if (nchunks > 1 && nchunks < 6 && (ngroups_all >> (nchunks + 1)) >= 2) ++nchunks;   // one more, smaller, tail chunk
    return nchunks;
}

cudaError_t mma_reserve_deferred(Plan *p, int64_t need)
{
    if (need <= p->cap_deferred) return cudaSuccess;
    if (p->d_deferred) cudaFree(p->d_deferred);
    p->d_deferred = nullptr; p->cap_deferred = 0;
    cudaError_t e = cudaMalloc(&p->d_deferred, (size_t)need * 4);
    if (e != cudaSuccess) return e;
    p->cap_deferred = need;
    return cudaSuccess;
}

cudaError_t mma_reserve_for(Plan *p, int64_t M)
{
    if (M <= 0) return cudaSuccess;
    // M * (nchunks(M) + 1) + 1 is not monotone in M below sm_count * 8 (where nchunks drops to 1): take the maximum
    const int64_t nc = p->specs.n_classes;
    int64_t need = nc * M * (mma_nchunks_for(p, M) + 1) + 1;
    for (int64_t m = 1; m <= std::min<int64_t>(M, (int64_t)p->sm_count * 8); ++m)
        need = std::max(need, nc * m * (mma_nchunks_for(p, m) + 1) + 1);
    return mma_reserve_deferred(p, need);
}

cudaError_t launch_signature_mma(Plan *p, const float *centres, int64_t M, float *sig, uint32_t *counts, cudaStream_t st)
{
    if (M == 0) return cudaSuccess;
    const int nchunks = mma_nchunks_for(p, M);
    const int slots_per_group = 128 / mma_nb_for(p->B);
    // deferred list: ROIs too large (<= M) + fix-list overflows (<= 1 per CTA).  Grown here only when apx_plan_reserve
    // has not sized it already (cudaFree / cudaMalloc synchronise the device: reserve first to keep apx_query asynchronous)
    cudaError_t e = mma_reserve_deferred(p, p->specs.n_classes * M * (nchunks + 1) + 1);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(p->d_deferred, 0, 4, st);
    if (e != cudaSuccess) return e;

    MmaParams q;
    q.sorted = p->d_sorted; q.cell_start = p->d_cell_start; q.grid = p->d_grid; q.centres = centres;
    q.dirs_sorted = p->d_dirs_sorted; q.perm = p->d_dir_perm; q.perm_mirror = p->mma_paired ? p->d_dir_perm_mirror : nullptr;
    q.table = reinterpret_cast<const uint4 *>(p->d_mma_table); q.phase = p->d_mma_phase; q.zeros = p->d_mma_zero;
    q.sig = reinterpret_cast<float2 *>(sig); q.counts = counts; q.deferred = p->d_deferred;
    q.hist_out = p->dbg_hist_out; q.hist_d0 = p->dbg_d0; q.hist_nd = p->dbg_nd;
#ifdef APX_TRACE
    q.trace = p->dbg_trace; q.trace_block = p->dbg_trace_block; q.trace_cap = p->dbg_trace_cap;
#endif
    q.ss = p->specs; q.norm0 = p->specs.norm[0];
    q.D = p->D; q.B = p->B; q.k_lo = p->k_lo; q.W = p->W; q.N = mma_n_for(p->W);
    q.nl = 0;
    while ((8 << q.nl) < p->B) ++q.nl;
    q.cap = mma_cap_for(p->B, q.N, p->W);
    const MmaSmem L0 = mma_smem_layout(p->B, q.N, p->W, q.cap);
    q.cap_big = L0.hist1 == L0.hist0 ? q.cap : std::min(8192, q.cap + (int)(L0.hist_bytes / 12));
    q.ngroups = p->Dp / slots_per_group;
    q.nchunks = nchunks;
    q.M = (int)M;
    q.clamp = p->need_clamp;
    q.half = p->mma_paired;
    q.unit_split = p->tune_unit_split;
    // a spare accumulator column (N > 4 W) carries the DC check, which lets a ROI of more than 2048 ions be binned in ONE pass
    q.dc_col = (q.N > 4 * q.W && p->tune_dc) ? 4 * q.W : -1;
    q.pass_ions = q.dc_col >= 0 ? (1 << 20) : 2048;
    q.nacc = (p->tune_nacc == 4 && 4 * q.N <= 512) ? 4 : 2;
    q.nacc_log2 = q.nacc == 4 ? 2 : 1;
    uint32_t cols = 32;
    while (cols < (uint32_t)(q.nacc * q.N)) cols *= 2;
    q.tmem_cols = cols;
    q.R = p->R; q.R2 = p->R2;
    const MmaSmem L = mma_smem_layout(p->B, q.N, p->W, q.cap);
    const int64_t blocks = M * nchunks;
    if (blocks > 0x7FFFFFFFLL) return cudaErrorInvalidConfiguration;
    auto launch = [&](auto kern) -> cudaError_t {
        cudaError_t le = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total);
        if (le != cudaSuccess) return le;
        kern<<<(unsigned)blocks, kMmaThreads, L.total, st>>>(q);
        return cudaSuccess;
    };
    const bool multi = p->specs.n_specs > 1;
    auto pick = [&](auto half_tag, auto multi_tag) -> cudaError_t {
        constexpr bool H = decltype(half_tag)::value, Mu = decltype(multi_tag)::value;
        if (p->B == 2048) return launch(k_signature_mma<16, 8, H, Mu>);
        if (p->B == 1024) return launch(k_signature_mma<16, 4, H, Mu>);
        if (p->B == 512) return launch(k_signature_mma<8, 4, H, Mu>);
        return launch(k_signature_mma<4, 4, H, Mu>);
    };
    if (p->mma_paired) e = multi ? pick(std::true_type{}, std::true_type{}) : pick(std::true_type{}, std::false_type{});
    else e = multi ? pick(std::false_type{}, std::true_type{}) : pick(std::false_type{}, std::false_type{});
    if (e != cudaSuccess) return e;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_signature_fft_list(p, centres, p->d_deferred, M, sig, counts, st);
}

}  // namespace apx
