/* hough_debug.h -- host-side introspection of libhough_b200.so.  NOT part of the product ABI
 * (include/hough.h); exported so that the CPU tests (tests/test_planner.py) can check, without a GPU, every
 * invariant of the launch shape and shared-memory layout the kernel relies on (DESIGN.md sections 4 and 5)
 * and emulate the voting loop's address arithmetic over every reachable bit pattern. */
#ifndef HOUGH_B200_DEBUG_H
#define HOUGH_B200_DEBUG_H

#ifdef __cplusplus
extern "C" {
#endif

/* The launch shape and shared-memory layout the library would choose for an n_theta x n_rho accumulator of
 * `acc_dtype` (HOUGH_ACC_*), with `cluster_size` / `ctas_per_sm` as in hough_set_option (0 = automatic) on a
 * device with `smem_optin` bytes of opt-in shared memory per CTA (0 = B200's 232448).  Needs NO CUDA device.
 * Writes HOUGH_PLAN_N_FIELDS values to out[] in the order of enum hough_plan_field; n_out must be at least
 * that.  Returns 0, HOUGH_ERR_INVALID_ARG, or HOUGH_ERR_UNSUPPORTED if nothing fits. */
enum { HOUGH_PLAN_N_FIELDS = 27 };
typedef enum hough_plan_field {
    HOUGH_PLAN_CLUSTER_SIZE = 0, HOUGH_PLAN_THREADS, HOUGH_PLAN_SMEM_BYTES, HOUGH_PLAN_ACC_BITS, HOUGH_PLAN_COLS_PER_LANE,
    HOUGH_PLAN_COLS_PER_CTA, HOUGH_PLAN_N_GROUPS, HOUGH_PLAN_N_STRIPES, HOUGH_PLAN_PITCH_BYTES, HOUGH_PLAN_BITMAP_WORDS_PER_ROW,
    HOUGH_PLAN_CHUNK_HITS, HOUGH_PLAN_REGION_BYTES, HOUGH_PLAN_PBM_OFF, HOUGH_PLAN_PBM_BYTES, HOUGH_PLAN_HB_OFF, HOUGH_PLAN_MISC_OFF,
    HOUGH_PLAN_W8_OFF, HOUGH_PLAN_W8_PITCH, HOUGH_PLAN_MCF_OFF, HOUGH_PLAN_MSF_OFF, HOUGH_PLAN_COLQ_OFF, HOUGH_PLAN_STASH_OFF,
    HOUGH_PLAN_CNT_OFF, HOUGH_PLAN_GCNT_OFF, HOUGH_PLAN_RCP_GROUPS, HOUGH_PLAN_RCP_2S, HOUGH_PLAN_CIRC_CAP
} hough_plan_field;
int hough_plan_describe(int n_theta, int n_rho, int acc_dtype, int cluster_size, int ctas_per_sm, int smem_optin,
                        long long* out, int n_out);

/* The two bounds that make a hit "tame" (eligible for the packed fast voting path) for
 * an n_rho-bin grid over +-rho_max and a trig table whose largest magnitude is `table_max` and smallest
 * non-zero magnitude `table_min_nz`, exactly as the kernel receives them: out2[0] = tame_bound (|u|+|v| must
 * not exceed it), out2[1] = ftz_min (u and v must each be 0 or at least this large in magnitude).  Host-only. */
int hough_debug_tame_bounds(int n_rho, float rho_max, float table_max, float table_min_nz, float* out2);

/* 1 if this library was built with -DHOUGH_DEBUG_BOUNDS (every shared-memory offset is checked; a violating
 * access is skipped and the event's d_counts becomes {-2, bit mask of the violating phases}), else 0. */
int hough_debug_bounds_enabled(void);

#ifdef __cplusplus
}
#endif
#endif /* HOUGH_B200_DEBUG_H */
