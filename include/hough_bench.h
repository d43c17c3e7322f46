/* hough_bench.h -- measurement aids of the B200 conformal Hough path.  NOT part of the product ABI
 * (include/hough.h): these calls live in a separate library, libhough_bench.so, that only bench.py, the
 * profiling commands under profiles/ and the GPU tests of the aids themselves load.  They give the
 * denominator of the vote roofline ("there is no published
 * shared-atomic peak for sm_100, the denominator is measured on the box") and the issue cost of the voting
 * loop's instructions ("dominant operations are regular multiply-add and index-mapping"). */
#ifndef HOUGH_B200_BENCH_H
#define HOUGH_B200_BENCH_H

#ifdef __cplusplus
extern "C" {
#endif

/* Times a kernel that does nothing but no-return 32-bit shared atomic adds (one accumulator
 * update per vote), `ctas_per_sm` x `threads` resident per SM on every SM, `iters` loop trips of 8 atomics per
 * thread, and returns atomics per second over the whole device in *out_rate.
 *   variant 0: every lane its own bank, add of 1 (ATOMS.POPC.INC), address arithmetic in the loop
 *   variant 1: every lane its own bank, add of a register value (ATOMS.ADD)
 *   variant 2: pseudo-random bank per lane (natural bank conflicts: the ceiling of a hit-per-lane mapping)
 *   variant 5: the ATOMS pipe alone: eight fixed conflict-free addresses per thread, no address arithmetic in
 *              the loop -- THE PEAK THE VOTE ROOFLINE DIVIDES BY
 * Synchronises the device.  Returns 0 or a negative code (-1 bad argument, -3 CUDA error, -4 out of memory). */
int hough_bench_shared_atomics(int variant, int ctas_per_sm, int threads, long long iters, double* out_rate);

/* The voting loop's instruction sequence (S2: six separately rounded fp32 operations per (hit, theta)
 * pair, row address, clamp, shared atomic) over a synthetic (u,v) buffer in the 180 x 256 u16 geometry (192
 * padded columns, 384-byte rows), with one instruction class removed or replaced at a time.  `mode` bits:
 *   1 = shared atomics issued (else the addresses are xor-reduced into a register)
 *   2 = clamp to the trash row (VIMNMX)         4 = IMAD row address (else a plain IADD of the lane offset)
 *   8 = packed fp32x2 arithmetic (else scalar)
 * `cpl` = theta columns per lane (2 or 6).  Returns lane-votes per second (padded lanes included) in *out_rate. */
int hough_bench_vote_loop(int mode, int cpl, int ctas_per_sm, int threads, long long iters, double* out_rate);

/* Issue rate of ONE instruction class (or a 1:1 mix of two), every warp of every SM running `iters` trips of an
 * unrolled block of 32 independent instructions; returns warp-instructions per second in *out_rate.
 * build.py checks the SASS of every kind: the loop body must hold exactly the named instructions.
 *   kind 0 FMUL   1 FADD   2 FFMA   3 FMUL2 (packed)   4 FADD2 (packed)   5 IMAD   6 VIMNMX (min.u32)
 *        7 IADD3  8 LOP3   9 LEA    10 FMUL+VIMNMX   11 FMUL+IMAD   12 FMUL2+VIMNMX   13 FMUL+IADD3 */
int hough_bench_issue_rate(int kind, int ctas_per_sm, int threads, long long iters, double* out_rate);

#ifdef __cplusplus
}
#endif
#endif /* HOUGH_B200_BENCH_H */
