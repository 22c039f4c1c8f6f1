/* aptsig_peaks.h -- C ABI of the on-chip peak microbenchmarks shipped inside libaptsig.so.
 *
 * SURVEY.md 8(d) bounds the project-and-bin step (Eq. 1) by plain FP32 issue and by
 * shared-memory atomic throughput, and the ion broadcast by shared-memory load throughput.  None of these
 * denominators is in MEASURED_PEAKS.json (HBM and bf16 tensor only), so the library measures them itself:
 * `python bench.py --peaks` runs every test below on the GPU and writes profiles/r2_peaks.json, which the
 * bench line's `roofline.peak` then cites.
 *
 * Each test launches one CTA of 1024 threads per SM; every warp issues the test's instruction
 * iters * 16 times with independent operands.  No device memory is touched in the timed loop.
 */
#ifndef APTSIG_PEAKS_H_
#define APTSIG_PEAKS_H_

#ifdef __cplusplus
extern "C" {
#endif

enum {
    APX_PEAK_FFMA = 0,                 /* fma.rn.f32: 2 flop per lane                                        */
    APX_PEAK_FFMA2 = 1,                /* fma.rn.f32x2 (packed pair, sm_100): 4 flop per lane                 */
    APX_PEAK_RED_CONFLICT_FREE = 2,    /* red.shared.add.u32, the 32 lanes on 32 different banks              */
    APX_PEAK_RED_2WAY = 3,             /* ... lanes l and l+16 on the same bank, different words              */
    APX_PEAK_RED_SAME_ADDRESS = 4,     /* ... all 32 lanes on one word                                        */
    APX_PEAK_RED_RANDOM_BANK = 5,      /* ... every lane on a random word of a 1.5 KB region                  */
    APX_PEAK_LDS32_BROADCAST = 6,      /* ld.shared.f32, one address per warp                                 */
    APX_PEAK_LDS32_CONFLICT_FREE = 7,  /* ld.shared.f32, 32 consecutive words                                 */
    APX_PEAK_LDS128_BROADCAST_1 = 8,   /* ld.shared.v4.f32, one address per warp                              */
    APX_PEAK_LDS128_BROADCAST_2 = 9,   /* ... one address per half-warp (the binning loop's ion load, B<=1024) */
    APX_PEAK_LDS128_BROADCAST_4 = 10,  /* ... one address per quarter-warp (B = 2048)                         */
    APX_PEAK_LDS128_CONFLICT_FREE = 11,/* ... 32 consecutive 16-byte words = 512 B per instruction            */
    APX_PEAK_RED_INC_CONFLICT_FREE = 12,/* red.shared.add.u32 of the literal 1 (ATOMS.POPC.INC), 32 banks; tests 2-5 add a
                                          register value (ATOMS.ADD)                                             */
    APX_PEAK_RED_SCATTERED_CONFLICT_FREE = 13, /* 32 different banks, every lane in a different 128-byte row: the access
                                          pattern of project-and-bin (a lane's row is its bin), the roofline denominator   */
    APX_PEAK_RED_SCATTERED_HALVES = 14,/* the kernel's bank map: lanes 0-15 on banks {0-3,8-11,16-19,24-27}, lanes 16-31 on
                                          the other sixteen, rows scattered                                           */
    APX_PEAK_COUNT = 15
};

typedef struct {
    int sm_count;                      /* CTAs launched = SMs of the device                                   */
    float ms;                          /* CUDA-event time of the timed launch                                 */
    double median_cycles;              /* clock64() ticks of the median CTA's timed loop                      */
    double warp_inst_per_s;            /* warp-level instructions of the test per second, whole GPU           */
    double warp_inst_per_clk_per_sm;   /* ... per SM clock and SM (median CTA)                                */
    double sm_mhz_effective;           /* median_cycles / ms: the SM clock the test actually ran at           */
} apx_peak_result;

/* Name of test `test` (static string), or NULL when test is out of range. */
const char *apx_peak_name(int test);

/* Run test `test` on CUDA device `device` with `iters` loop iterations (16 instructions each) per warp;
 * `out` is a HOST pointer.  Synchronises the device.  Returns 0, -1 (bad argument) or -3 (CUDA error). */
int apx_peak_measure(int device, int test, int iters, apx_peak_result *out);

#ifdef __cplusplus
}
#endif
#endif /* APTSIG_PEAKS_H_ */
