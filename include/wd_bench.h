/* include/wd_bench.h — C-ABI of libwdbench: measurement helpers that bench.py uses for the roofline
 * denominators.  NOT part of the product library (libwd.so exports none of these).
 */
#ifndef WD_BENCH_H
#define WD_BENCH_H

#ifdef __cplusplus
extern "C" {
#endif

/* Register-only FP64 FMA microbenchmark (the paper's section 3.1 method): the FP64 roof that
 * co-limits a multi-RHS application.  Launches threads_per_sm-thread CTAs (a multiple of 32, <= 1024) filling
 * every SM (one_cta_per_sm = 0) or exactly one per SM (1), each thread running `ilp` (1, 2, 4, 8, 16) independent
 * FMA chains; distinct_operands = 0: a = fma(a, b, c) with b, c common to all chains, 1: every operand of every
 * chain a register pair of its own.  *tflops = achieved 2*FMA/s; *cycles_per_fma_per_warp (may be NULL) = cycles
 * of the nominal maximum SM clock between two FMAs issued on one SM sub-partition.  Synchronous, default stream.
 * Returns 0, or a negative code (-1 bad argument, -2 out of memory, -4 CUDA error). */
int wdb_measure_fp64(int threads_per_sm, int ilp, int one_cta_per_sm, int distinct_operands, double *tflops,
                     double *cycles_per_fma_per_warp);

/* Streaming ceilings of the device memory ("also measure a read-only streaming
 * ceiling"): a grid-stride kernel over `bytes` of device memory (allocated inside, > L2), best of `reps`.
 * mode 0: read only (LDG.128, sum kept in registers); 1: copy (read + write, the mix of MEASURED_PEAKS.json);
 * 2: 7 reads : 1 write, the mix of one Wilson-clover application (1344 B read, 192 B written per site).
 * *gbs = bytes moved (reads + writes) / time. */
int wdb_measure_stream(int mode, size_t bytes, int reps, double *gbs);

/* What an LDS.128 costs for a given lane-to-address pattern: the measurement behind the lane mapping of the quad
 * multi-RHS kernels (csrc/wd_tmq.cu).  One CTA of 256 threads per SM issues back-to-back
 * LDS.128; *cycles = SM cycles per warp instruction (the pipe moves 128 B per cycle, so 4.0 = 512 distinct bytes).
 * pattern 0: every lane its own 16 bytes (512 B per warp)
 *         1: lane & 7   — the same 128 bytes in each quarter-warp   (lane = r * 8 + site: links of the plain layout)
 *         2: lane >> 2  — one address per four ADJACENT lanes        (lane = site * 4 + r: links of the blocked layout)
 *         3: all lanes one address
 *         4: four 128-byte-aligned segments, segment = lane & 3       (psi with lane = site * 4 + r on the plain layout)
 *         5: four segments, segment = lane >> 3                       (psi with lane = r * 8 + site)
 *         6: lane >> 1  — one address per pair of adjacent lanes */
int wdb_measure_lds(int pattern, double *cycles);

#ifdef __cplusplus
}
#endif
#endif /* WD_BENCH_H */
