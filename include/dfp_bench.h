/* dfp_bench.h - C ABI of libdfp_bench.so: micro-benchmarks that MEASURE the denominators of the roofline of the dfp
 * projector kernels.  A probe for bench.py, NOT part of the method and not part of libdfp.so (include/dfp.h).
 *
 * The projector kernels are bound by the SM-side pipes and not by HBM.
 * dfp_microbench runs one resident wave of a small kernel on the current device (default stream, synchronous, timed
 * with CUDA events, allocates and frees a few MB of scratch) and writes the sustained rate of the WHOLE DEVICE PER
 * SECOND (divide by SM count x SM clock for the rate per clock per SM):
 *   DFP_MB_LDS   warp-wide, bank-conflict-free LDS.32 instructions (the staged gradient kernels need 32 per
 *                warp-sample and 12 per warp-voxel-view);
 *   DFP_MB_FADD / DFP_MB_FFMA / DFP_MB_FFMA2   fp32 results of dependent-free FADD, FFMA and packed FFMA2 streams.
 * kind: one of DFP_MB_*; per_second: host pointer, out.  Returns DFP_BENCH_OK, DFP_BENCH_ERR_NULL (per_second is NULL),
 * DFP_BENCH_ERR_KIND (unknown kind) or DFP_BENCH_ERR_CUDA (no device / runtime failure).
 */
#ifndef DFP_BENCH_H_
#define DFP_BENCH_H_

#ifdef __cplusplus
extern "C" {
#endif

enum { DFP_MB_LDS = 0, DFP_MB_FADD = 1, DFP_MB_FFMA = 2, DFP_MB_FFMA2 = 3 };
enum { DFP_BENCH_OK = 0, DFP_BENCH_ERR_NULL = -1, DFP_BENCH_ERR_KIND = -2, DFP_BENCH_ERR_CUDA = -6 };

int dfp_microbench(int kind, double* per_second);

#ifdef __cplusplus
}
#endif
#endif /* DFP_BENCH_H_ */
