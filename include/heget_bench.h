/* heget_bench.h -- entry points of libheget.so that are NOT part of the product surface of
 * include/heget.h: the roofline denominators and the launch counter bench.py reports, and the
 * paper's own List 2 program as a same-GPU comparison.  Same conventions as heget.h.
 * Citations are PAPER.md line numbers. */
#ifndef HEGET_BENCH_H
#define HEGET_BENCH_H

#include "heget.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Peak-rate microbenchmark used for the roofline denominator: launches a kernel of
 * independent FMA chains (precision = HEGET_FP32 / HEGET_FP64) filling every SM and
 * writes the achieved FLOP/s (FMA = 2) to *flops_per_s [host].  Synchronises. */
int heget_fma_peak(heget_ctx* ctx, int precision, double* flops_per_s);

/* The same measurement for other operand patterns (context for the roofline: the amplitude
 * kernels' FMAs take three register operands, which the register file cannot feed at the
 * pipe's peak rate):
 *   HEGET_PEAK_CONST_OPERAND  x = x*a + b, a and b constant-bank operands (= heget_fma_peak)
 *   HEGET_PEAK_THREE_REG      x = y*z + x, three distinct registers, no operand reuse
 *   HEGET_PEAK_NODE_PATTERN   the fvixx0 node (16 FMA + 4 MUL per node, 36 flop) on registers */
enum { HEGET_PEAK_CONST_OPERAND = 0, HEGET_PEAK_THREE_REG = 1, HEGET_PEAK_NODE_PATTERN = 2 };
int heget_fma_peak_pattern(heget_ctx* ctx, int precision, int pattern, double* flops_per_s);

/* Number of kernel launches this context has issued (all entry points), for bench.py's
 * gpu_launches count. */
int64_t heget_launch_count(const heget_ctx* ctx);

/* The paper's own program, List 2 generalised to n photons, run the way the
 * paper runs it: one thread per event, one drawn helicity assignment per event, 4-component HEGET
 * functions on cmplx w[6] (ixxxx1, oxxxx2, vxxxx0, n-1 fvoxx0 chained from the ubar line and one
 * iovxxx per permutation, iPNext through the n! orderings), no prefix reuse, no tables.  Same
 * arguments, helicity draw and result as heget_amp2_sampled (4 * 2^n * |M(h_e)|^2): it is the
 * design this library is measured against on the same GPU. */
int heget_list2(heget_ctx* ctx, uint64_t seed, uint64_t first_event, const double* momenta, int n,
                int precision, double* out_amp2, int32_t* out_hel, int64_t N, void* stream);

/* The same program called for every one of the 4 * 2^n helicity assignments inside the thread:
 * out_amp2[e] = sum |M|^2, the quantity heget_amp2 returns, computed with the paper's arithmetic
 * (no prefix reuse, no parity, 4-component; SURVEY 8(d) model A).  A same-GPU baseline for the
 * headline metric; n = 7, 8 take minutes per 10^4 events. */
int heget_list2_sum(heget_ctx* ctx, const double* momenta, int n, int precision, double* out_amp2,
                    int64_t N, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* HEGET_BENCH_H */
