/* hough.h -- C ABI of the B200-native conformal-mapped, matrix-form Hough
 * transform (arxiv/paper_2607_04067; citations are PAPER.md line numbers).
 *
 * What the library computes, per event, entirely on the GPU (one fused kernel
 * launch per hough_run call):
 *   H0/H1  load the event's hits P = {(x_i, y_i)} and map them to
 *          the conformal plane, u = x/(x^2+y^2), v = y/(x^2+y^2)  (Eq. (1));
 *   H2     rho_ij = u_i cos(theta_j) + v_i sin(theta_j) for the shared theta
 *          table, the matrix R of PAPER.md:92-96, binned at equal intervals
 *          over [-rho_max, rho_max);
 *   H3     vote every in-range (hit, theta_j) pair into the event's
 *          N_theta x N_rho integer accumulator, held in shared memory
 *          (block-local accumulation);
 *   H4/H5  threshold + 3x3 local-maximum peaks, listed in raster order
 *          (peak finding + NMS on the device);
 *   H6     keep every hit whose own (theta, rho) bins fall inside any stored
 *          peak's +-window (the hit filter of PAPER.md:44, :75);
 *   H7     stable per-event compaction of the kept hits (N_select of Eq. (8),
 *          PAPER.md:118-123).
 * Arithmetic: fp32, round-to-nearest-even, one rounding per operation (no FMA
 * contraction), IEEE division, denormals kept; integer results are exact.
 * The exact operation order is DESIGN.md "Readings" S1-S6.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The
 *     caller owns every buffer it passes; the library owns only the handle,
 *     its device copy of the cos/sin table and (for hough_run_host only) a
 *     grow-only device staging area.
 *   - hough_run / hough_run_ex are asynchronous on `stream`: they never
 *     synchronise, never allocate, never read device data on the host, keep no
 *     per-run scratch (one handle may be used from several streams at once)
 *     and can be captured in a CUDA graph.
 *   - All functions return 0 on success or a negative hough_status.
 *   - There is no CPU fallback: without a CUDA device every call fails with
 *     HOUGH_ERR_CUDA.
 */
#ifndef HOUGH_B200_H
#define HOUGH_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hough_ctx hough_ctx;      /* opaque, library-owned */
typedef void* hough_stream;              /* a cudaStream_t (CUstream); NULL = default stream */

/* One peak (H5): accumulator cell (theta_bin, rho_bin) and its vote count. 8 bytes. */
typedef struct hough_peak {
    uint16_t theta_bin;
    uint16_t rho_bin;
    uint32_t votes;
} hough_peak;

/* Candidate circle and track parameters of one stored peak (hough_circles; Eq. (2)). 48 bytes.
 * Lengths in the units of the hit coordinates; pt in GeV/c when those are mm and the field is in tesla. */
typedef struct hough_circle {
    double x_c, y_c, r_c;   /* centre and radius of the circle through the origin */
    double pt;              /* 0.3 B r_c */
    double phi0;            /* direction of motion at the origin, [0, 2 pi) */
    int32_t charge;         /* +1 / -1 turning sense from the associated hits, 0 when undecided */
    int32_t n_hits;         /* hits associated with the peak */
} hough_circle;

typedef enum hough_status {
    HOUGH_OK = 0,
    HOUGH_ERR_INVALID_ARG = -1,   /* null pointer, out-of-range value */
    HOUGH_ERR_UNSUPPORTED = -2,   /* grid does not fit even a 16-CTA cluster's shared memory */
    HOUGH_ERR_CUDA = -3,          /* a CUDA call failed (no device, launch error, ...) */
    HOUGH_ERR_NOMEM = -4          /* host or device allocation failed */
} hough_status;

typedef enum hough_option {
    HOUGH_OPT_MAX_PEAKS = 1,        /* peaks stored per event, 0..1048576 (default 64) */
    HOUGH_OPT_ACC_DTYPE = 2,        /* HOUGH_ACC_AUTO (= u16), HOUGH_ACC_U16, HOUGH_ACC_U32 */
    HOUGH_OPT_CONFORMAL_SCALE = 3,  /* 1 (Eq. (1) as printed, default) or 2 (the scale Eq. (2) implies) */
    HOUGH_OPT_CLUSTER_SIZE = 4,     /* 0 = smallest of {1,2,4,8,16} that fits (default), else force one of them; 16 is a
                                       non-portable cluster size, taken only when nothing smaller fits (the paper's own
                                       1000 x 1000 grid) */
    HOUGH_OPT_CTAS_PER_SM = 5,      /* 0 = as many as fit, up to 2 (default); tuning knob */
    HOUGH_OPT_VOTE_PATH = 6,        /* 0 = fast voting with packed fp32x2 arithmetic, the exact slow path only for
                                       degenerate hits (default); 1 = force the exact slow path everywhere (testing) */
    /* Variants of the paper's own wording (readings Q18-Q20).  Any non-default
       value selects the extended instantiation of the kernel; the defaults run the instantiation bench.py times. */
    HOUGH_OPT_PEAK_MODE = 7,        /* 0 = absolute threshold + 3x3 local maximum, raster order (default);
                                       1 = threshold relative to the event's global accumulator maximum + iterative
                                       "extract the most significant peak, suppress its neighbourhood":
                                       peaks come out in extraction order (descending votes) */
    HOUGH_OPT_REL_THRESHOLD_PERMILLE = 8,  /* peak mode 1: candidates need votes >= ceil(value * A_max / 1000) and >= threshold;
                                       0..1000, default 500 */
    HOUGH_OPT_NMS_RADIUS = 9,       /* peak mode 1: half-width in bins of the suppressed neighbourhood, 0..64 (default 1) */
    HOUGH_OPT_THETA_WRAP = 10,      /* 1 = (theta + pi, rho) == (theta, -rho): column -1 is column n_theta-1 with the rho
                                       index mirrored, for the 3x3 test, the suppression and the keep windows (default 0) */
    HOUGH_OPT_KEEP_MODE = 11,       /* 0 = (theta, rho) window around the stored peaks (default); 1 = original-space road
                                       | ||hit - centre|| - r_c | < HOUGH_OPTF_KEEP_TOL around their candidate circles
                                       ("inversely mapped back to the original space ... data filtering") */
    HOUGH_OPT_STAGING = 12,         /* how an event's hits reach shared memory (H0; PAPER.md:86 names non-coalesced access
                                       as a hazard): 0 = coalesced float2 loads issued ahead of the zeroing stores (default);
                                       1 = one cp.async.bulk (TMA engine) per chunk, completion on an mbarrier, the 16-byte
                                       aligned source range found by aligning down and up by one hit; needs d_xy 16-byte
                                       aligned.  Same results; never yet timed */
    HOUGH_OPT_SCHEDULER = 13,       /* how events reach the SMs (events "assigned to different thread blocks"):
                                       0 = one CTA (cluster) per event, dealt by the hardware block scheduler (default);
                                       1 = the same launch, but a resident CTA cancels the launch of a not-yet-started CTA
                                       (Blackwell cluster launch control) and takes over its event, so the per-CTA set-up
                                       runs once per resident CTA, and the next event's hits are prefetched into L2 under
                                       the current event's peak finding and selection; one-CTA-per-event grids only (a
                                       clustered grid ignores it); needs d_xy 16-byte aligned.  Same results; never yet timed */
    HOUGH_OPT_SELECT_MODE = 14      /* how H6 finds the hits inside a stored peak's window (same result):
                                       0 = every hit scans the MARKED theta columns, one thread per hit (default; cheap when
                                       few columns are marked);
                                       1 = dense: the dead accumulator is rewritten as the window mask and every hit is
                                       tested at ALL columns with the voting loop's own mapping (lane = column, packed
                                       arithmetic, conflict-free loads, one ballot per hit): one voting-sized pass whatever
                                       the number of peaks;
                                       2 = dense when the stored peaks' windows could cover more than half of the columns.
                                       One-CTA-per-event grids with the window filter only (a clustered grid, the distance
                                       filter, or an event with more hits than the peak bitmap has bits keep mode 0).
                                       Never yet timed */
} hough_option;

typedef enum hough_option_f64 {
    HOUGH_OPTF_KEEP_TOL = 1,        /* keep mode 1: road half-width, units of the hit coordinates, >= 0 (default 0) */
    HOUGH_OPTF_B_FIELD_TESLA = 2    /* hough_circles: magnetic field for pt = 0.3 B r_c (default 1.0) */
} hough_option_f64;

enum { HOUGH_ACC_AUTO = 0, HOUGH_ACC_U16 = 1, HOUGH_ACC_U32 = 2 };

typedef enum hough_info {
    HOUGH_INFO_CLUSTER_SIZE = 1,    /* CTAs per event */
    HOUGH_INFO_THREADS = 2,         /* threads per CTA */
    HOUGH_INFO_SMEM_BYTES = 3,      /* dynamic shared memory per CTA */
    HOUGH_INFO_CTAS_PER_SM = 4,     /* resident CTAs per SM (occupancy query) */
    HOUGH_INFO_GRID_MAX = 5,        /* CTAs resident on the device at once (a launch has one CTA or cluster per event) */
    HOUGH_INFO_ACC_BITS = 6,        /* 16 or 32 */
    HOUGH_INFO_MAX_PEAKS = 7,
    HOUGH_INFO_CHUNK_HITS = 8,      /* hits staged in shared memory per pass */
    HOUGH_INFO_SM_COUNT = 9,
    HOUGH_INFO_LAUNCHES = 10        /* kernels launched through this handle so far */
} hough_info;

/* Creates a handle for an n_theta x n_rho accumulator over theta in [0, pi)
 * (theta_j = j*pi/n_theta) and rho in [-rho_max, rho_max)
 * (rho_max in 1/units of the hit coordinates), an absolute vote threshold
 * (>= 1) and a keep window of +-window bins in theta and rho (>= 0).
 * Builds the default cos/sin table ((float)cos((double)j*pi/n_theta)) and
 * copies it to the device.  Requires 1 <= n_theta <= 65535, 1 <= n_rho <= 65535,
 * rho_max finite and > 0.  Returns NULL on failure; hough_last_error() says why. */
hough_ctx* hough_create(int n_theta, int n_rho, float rho_max, int threshold, int window);

/* Sets an option (see hough_option).  Must not be called while a run that uses
 * the handle is in flight.  HOUGH_ERR_UNSUPPORTED if the resulting
 * configuration does not fit the device. */
int hough_set_option(hough_ctx* ctx, int key, long long value);

/* Sets a real-valued option (see hough_option_f64). */
int hough_set_option_f64(hough_ctx* ctx, int key, double value);

/* Replaces the theta table of the rho matrix R ("discrete
 * angle theta_j", the cos/sin factors of PAPER.md:69): h_cos[j], h_sin[j],
 * j < n_theta, HOST pointers, copied (synchronously).  Values must be finite.
 * Lets a caller fix theta samples other than the default left bin edges
 * (the paper does not say edge or centre, reading Q3) and hands the
 * kernel the very table an external checker uses. */
int hough_set_trig_table(hough_ctx* ctx, const float* h_cos, const float* h_sin);

/* Reads a property of the current configuration (see hough_info); negative on error. */
long long hough_get_info(const hough_ctx* ctx, int key);

/* Runs H0-H7 on a batch (events are batched and independent).
 *   d_xy            [n_total][2] fp32, interleaved (x, y); event e's hits are
 *                   rows d_event_offsets[e] .. d_event_offsets[e+1]-1
 *   d_event_offsets [n_events+1] int32, non-decreasing (CSR); not validated,
 *                   decreasing offsets are undefined behaviour
 *   d_keep_mask     [n_total] u8, written 0/1 for every hit
 *   d_peaks         [n_events][max_peaks]; the first min(n_peaks, max_peaks)
 *                   entries of an event are written, in raster order
 *                   (theta_bin major, then rho_bin); the rest are untouched
 *   d_counts        [n_events][2] int32 = {n_peaks found (untruncated), n_kept}
 * An event with more than 65535 hits under a u16 accumulator gets counts
 * {-1,-1} and no other output.  n_events == 0 is a successful no-op. */
int hough_run(hough_ctx* ctx, const float* d_xy, const int32_t* d_event_offsets, int n_events,
              uint8_t* d_keep_mask, hough_peak* d_peaks, int32_t* d_counts, hough_stream stream);

/* hough_run plus optional outputs (any of the last three may be NULL): the
 * reduced hit set itself (the N_select hits of Eq. (8), that
 * go on to track fitting) and the accumulator of PAPER.md:96-104:
 *   d_kept_xy    [n_total][2] fp32 and
 *   d_kept_idx   [n_total] int32: event e's kept hits, in original order, start
 *                at d_event_offsets[e]; kept_idx is the index within the event;
 *                entries past n_kept are untouched
 *   d_accum_dump [n_events][n_theta][n_rho] u32: the accumulator (parity and
 *                debugging only; never part of a timed run) */
typedef struct hough_io {
    const float* d_xy;
    const int32_t* d_event_offsets;
    int32_t n_events;
    uint8_t* d_keep_mask;
    hough_peak* d_peaks;
    int32_t* d_counts;
    float* d_kept_xy;
    int32_t* d_kept_idx;
    uint32_t* d_accum_dump;
} hough_io;

int hough_run_ex(hough_ctx* ctx, const hough_io* io, hough_stream stream);

/* Candidate-circle and track-parameter extraction for the stored peaks of a finished hough_run on the same
 * stream: "the line in conformal space can be inversely mapped to the circular-track
 * parameters" (Eq. (2) at :77), pT and phi0 as evaluated at PAPER.md:150-158.  Per stored peak
 * (theta_j, rho bin k), in fp64 with one rounding per operation (readings Q14-Q17):
 *   rho_c = (k + 0.5)/inv - rho_max (bin centre);  centre = s (cos theta_j, sin theta_j) / (2 rho_c);
 *   r_c = s / (2 |rho_c|), s = the conformal scale (s = 2 is Eq. (2) as printed);  pt = 0.0003 B r_c;
 *   a hit is associated with the peak iff its own bin at column j is within the keep window of k; the side of the
 *   centre direction on which the associated hits lie gives the turning sense (charge) and
 *   phi0 = centre azimuth - charge * pi/2.
 *   d_peaks, d_counts  as written by hough_run for the same d_xy / d_event_offsets
 *   d_circles          [n_events][max_peaks] hough_circle; the first min(n_peaks, max_peaks) entries of an event are
 *                      written, the rest are untouched
 * One kernel launch, asynchronous on `stream`, no allocation, capturable. */
int hough_circles(hough_ctx* ctx, const float* d_xy, const int32_t* d_event_offsets, int n_events,
                  const hough_peak* d_peaks, const int32_t* d_counts, hough_circle* d_circles, hough_stream stream);

/* End-to-end form with HOST buffers (pinned memory recommended), the shape of
 * the paper's own measurement: events are "transmitted to the GPU memory" in
 * batches and "only the extracted peak results need to be returned"
 * (PAPER.md:90, :106).  Copies
 * h_xy / h_event_offsets to a library-owned device staging area, runs H0-H7
 * and copies keep mask, peaks and counts (and kept_xy / kept_idx when not
 * NULL) back, all asynchronously on `stream`; the host outputs are valid after
 * the caller synchronises `stream`.  h_kept_xy / h_kept_idx NULL = lean mode:
 * only mask, peaks and counts come back (a host consumer that still holds h_xy
 * can compact by the mask).  Only the entries hough_run defines are meaningful;
 * the rest of h_peaks and of the kept arrays is zero.
 *   The hit arrays (h_xy, h_keep_mask, h_kept_xy, h_kept_idx) are indexed by the
 * offsets themselves: a SUB-BATCH of a larger host array passes the same array
 * pointers with h_event_offsets advanced to its first event, and only its own
 * hits h_event_offsets[0] .. h_event_offsets[n_events]-1 are copied; h_peaks and
 * h_counts belong to the sub-batch ([n_events][...]).  The library keeps one
 * device staging area per stream (up to 8 streams at a time, grow-only), so
 * sub-batches issued on different streams overlap their host-to-device copy,
 * kernel and device-to-host copies.
 * Calls on ONE stream must not overlap in time from several host threads. */
int hough_run_host(hough_ctx* ctx, const float* h_xy, const int32_t* h_event_offsets, int n_events,
                   uint8_t* h_keep_mask, hough_peak* h_peaks, int32_t* h_counts,
                   float* h_kept_xy, int32_t* h_kept_idx, hough_stream stream);

/* Releases the handle and everything it owns.  NULL is allowed. */
void hough_destroy(hough_ctx* ctx);

const char* hough_strerror(int status);
const char* hough_last_error(void);      /* thread-local message of the last failure */
const char* hough_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HOUGH_B200_H */
