// hough_api.cu -- the C ABI of include/hough.h: handle management, shared-memory
// planning, launch.  All compute is in hough_kernel.cuh; nothing here falls
// back to the CPU.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "../../include/hough_debug.h"
#include "hough_kernel.cuh"

using hough::KParams;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(call)                                                                          \
    do {                                                                                        \
        cudaError_t _e = (call);                                                                \
        if (_e != cudaSuccess) return fail(HOUGH_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(_e)); \
    } while (0)

inline int align_up(int x, int a) { return (x + a - 1) / a * a; }

struct Plan {
    bool acc16 = true;
    int cpl = 2;             // theta columns per lane in the vote phase (kernel template parameter)
    int csize = 1;
    int threads = 0;
    int smem_bytes = 0;
    int ctas_per_sm = 0;     // measured with the occupancy API
    int grid_max = 0;
    KParams kp{};            // geometry part filled in; pointers per run
};

}  // namespace

// Device staging area of hough_run_host for one stream.
struct Staging {
    bool used = false;
    cudaStream_t stream = nullptr;
    unsigned long long tick = 0;
    long long cap_hits = 0, cap_peaks = 0;
    int cap_events = 0;
    float* xy = nullptr;
    int32_t* off = nullptr;
    uint8_t* keep = nullptr;
    hough_peak* peaks = nullptr;
    int32_t* counts = nullptr;
    float* kept_xy = nullptr;
    int32_t* kept_idx = nullptr;
    void release() {
        cudaFree(xy); cudaFree(off); cudaFree(keep); cudaFree(peaks); cudaFree(counts); cudaFree(kept_xy); cudaFree(kept_idx);
        xy = nullptr; off = nullptr; keep = nullptr; peaks = nullptr; counts = nullptr; kept_xy = nullptr; kept_idx = nullptr;
        cap_hits = 0; cap_peaks = 0; cap_events = 0;
    }
};

struct hough_ctx {
    int n_theta, n_rho, threshold, window;
    float rho_max, inv;
    int max_peaks = 64;
    int acc_dtype = HOUGH_ACC_AUTO;
    int conformal_scale = 1;
    int opt_cluster = 0;
    int opt_ctas_per_sm = 0;
    int opt_vote_path = 0;
    int peak_mode = 0, rel_permille = 500, nms_radius = 1, theta_wrap = 0, keep_mode = 0, stage_mode = 0, sched_mode = 0, select_mode = 0;
    double keep_tol = 0.0, b_field = 1.0;
    int device = 0;
    int sm_count = 0;
    int smem_optin = 0;
    float* d_cos = nullptr;
    float* d_sin = nullptr;
    float tmax = 1.0f;
    float tmin_nz = 1.0f;    // smallest non-zero magnitude in the trig table
    Plan plan;
    std::atomic<long long> launches{0};
    // hough_run_host staging: one grow-only device area per stream (up to 8 streams at a time)
    Staging staging[8];
    unsigned long long staging_tick = 0;
    std::mutex staging_mu;
};

namespace {

template <bool ACC16, bool CL, bool EXT>
const void* kernel_ptr(int cpl) {
    switch (cpl) {
        case 6: return (const void*)&hough::hough_event_kernel<ACC16, CL, 6, EXT>;
        case 4: return (const void*)&hough::hough_event_kernel<ACC16, CL, 4, EXT>;
        default: return (const void*)&hough::hough_event_kernel<ACC16, CL, 2, EXT>;
    }
}

// ext: the extended instantiation (peak mode, theta wrap, distance filter); the default options never take it, so the
// kernel bench.py times is compiled without any of that code.
const void* pick_kernel(bool acc16, bool cl, int cpl, bool ext) {
    if (ext) {
        if (acc16) return cl ? kernel_ptr<true, true, true>(cpl) : kernel_ptr<true, false, true>(cpl);
        return cl ? kernel_ptr<false, true, true>(cpl) : kernel_ptr<false, false, true>(cpl);
    }
    if (acc16) return cl ? kernel_ptr<true, true, false>(cpl) : kernel_ptr<true, false, false>(cpl);
    return cl ? kernel_ptr<false, true, false>(cpl) : kernel_ptr<false, false, false>(cpl);
}

bool wants_ext(const hough_ctx* c) { return c->peak_mode != 0 || c->theta_wrap != 0 || c->keep_mode != 0 || c->stage_mode != 0 || c->sched_mode != 0 || c->select_mode != 0; }

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel (per device), not to a handle: several live
// handles may share one instantiation with different footprints, so the attribute is only ever RAISED.
int raise_smem_limit(int device, const void* fn, int bytes) {
    static std::mutex mu;
    static std::map<std::pair<int, const void*>, int> high;
    std::lock_guard<std::mutex> lk(mu);
    int& h = high[std::make_pair(device, fn)];
    if (bytes <= h) return HOUGH_OK;
    CUDA_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    h = bytes;
    return HOUGH_OK;
}

// Launch attributes of the kernel this handle would launch now: shared-memory limit (raised, never lowered) and, for a
// 16-CTA cluster, the non-portable-cluster-size permission.
int prepare_kernel(int device, const void* fn, int smem_bytes, int csize) {
    if (int rc = raise_smem_limit(device, fn, smem_bytes)) return rc;
    if (csize > 8) CUDA_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    return HOUGH_OK;
}

// Lays out shared memory for cluster size C, `want_ctas` CTAs per SM and `cpl` theta columns per lane.  Returns false if
// it does not fit or an invariant of the kernel's address arithmetic cannot be met.
bool try_plan_cpl(const hough_ctx* c, bool acc16, int C, int want_ctas, int cpl, Plan* out) {
    const int cols = (c->n_theta + C - 1) / C;
    const int padded = (cols + 32 * cpl - 1) / (32 * cpl) * (32 * cpl);
    const int n_groups = padded / (32 * cpl);
    const int max_warps = want_ctas >= 2 ? 16 : 32;
    if (n_groups > max_warps) return false;
    const int pitch_b = n_groups * cpl * (acc16 ? 64 : 128);
    if (pitch_b > 8192) return false;
    const long long acc_bytes = ((long long)c->n_rho + 1) * pitch_b;   // + the trash row
    // Padding columns carry NaN table entries; their bins are the canonical NaN (0x7FFFFFFF) and must fall
    // beyond the accumulator after the wrapping multiply by the pitch, for every word offset of a row.
    {
        const unsigned nan_rel = (0x7FFFFFFFu - HOUGH_MAGIC_BITS) * (unsigned)pitch_b;
        const unsigned long long end = (unsigned long long)(c->n_rho + 1) * (unsigned)pitch_b;
        // (the largest lane offset added to it is pitch - 4: no 32-bit wrap back into the accumulator)
        if ((unsigned long long)nan_rel < end || (unsigned long long)nan_rel + (unsigned)pitch_b - 4ull > 0xFFFFFFFFull) return false;
    }
    const int wpr = (c->n_rho + 31) / 32;
    const int n_stripes = max_warps / n_groups;
    const int threads = 32 * n_groups * n_stripes;
    const int nwarps = threads / 32;
    // post-extraction data that reuses the accumulator region
    long long o = 0;
    KParams kp{};
    kp.w8_pitch = align_up(c->n_rho + 1, 16);          // byte n_rho of a row is the always-zero clamp target
    kp.w8_off = (int)o;      o += (long long)((c->n_theta + 7) / 8) * kp.w8_pitch;
    kp.mcf_off = (int)o;     o += align_up((c->n_theta + 8) * 4, 16);
    kp.msf_off = (int)o;     o += align_up((c->n_theta + 8) * 4, 16);
    kp.colq_off = (int)o;    o += align_up(c->n_theta * 4, 16);
    kp.stash_off = (int)o;   o += (C > 1) ? align_up(HOUGH_SEL_ROUND_BLOCKS * nwarps * 4, 16) : 0;
    kp.cnt_off = (int)o;     o += (C > 1) ? align_up(HOUGH_SEL_ROUND_BLOCKS * 4, 16) : 0;
    kp.gcnt_off = (int)o;    o += (C > 1) ? align_up((HOUGH_SEL_ROUND_BLOCKS * C + 1) * 4, 16) : 0;
    const long long post_bytes = o;
    const long long region = align_up((int)std::max(acc_bytes, o), 16);
    // the peak bitmap; iterative NMS (peak mode 1) keeps one 8-byte key per rho row there instead
    const long long pbm_bytes = std::max(align_up(cols * wpr * 4, 16), align_up(8 * c->n_rho, 16));
    const long long misc_bytes = 256;
    const long long fixed = region + pbm_bytes + misc_bytes;
    // per-CTA budget: the SM has 228 KB, each resident CTA reserves 1 KB; a single CTA may opt in to smem_optin
    long long budget = (long long)(233472 / want_ctas) - 1024;
    if (budget > c->smem_optin) budget = c->smem_optin;
    long long chunk = (budget - fixed) / 8;
    if (chunk < 128) return false;
    if (chunk > 4096) chunk = 4096;
    chunk &= ~1LL;
    kp.csize = C;
    kp.cols_per_cta = cols;
    kp.n_groups = n_groups;
    kp.n_stripes = n_stripes;
    kp.rcp_groups = 65536u / (unsigned)n_groups + 1u;
    kp.rcp_2s = (1u << 20) / (unsigned)(2 * n_stripes) + 1u;
    for (unsigned w = 0; w < 32; ++w)
        if (((w * kp.rcp_groups) >> 16) != w / (unsigned)n_groups) return false;
    for (unsigned m = 0; m <= (unsigned)chunk; ++m)
        if (((m * kp.rcp_2s) >> 20) != m / (unsigned)(2 * n_stripes)) return false;
    kp.vpr = pitch_b / 16;
    kp.pitch_b = pitch_b;
    kp.wpr = wpr;
    kp.chunk = (int)chunk;
    kp.region_bytes = (int)region;
    kp.pbm_off = (int)region;
    kp.pbm_bytes = (int)pbm_bytes;
    kp.hb_off = (int)(region + pbm_bytes);
    // distance filter: (x_c, y_c, r_c) doubles staged from the start of the dead accumulator region, in a cluster up to
    // the compaction scratch (stash/cnt/gcnt live there at the same time)
    kp.circ_cap = (int)(((C > 1 ? (long long)kp.stash_off : region) - kp.w8_off) / 24);
    (void)post_bytes;
    kp.misc_off = kp.hb_off + (int)chunk * 8;
    out->acc16 = acc16;
    out->cpl = cpl;
    out->csize = C;
    out->threads = threads;
    out->smem_bytes = kp.misc_off + (int)misc_bytes;
    out->kp = kp;
    return true;
}

// Columns per lane: the choice that pads the fewest columns first, ties to the larger (fewer broadcast loads per
// vote); a choice whose row pitch breaks an address invariant (e.g. the NaN rule above) falls through to the next.
bool try_plan(const hough_ctx* c, bool acc16, int C, int want_ctas, Plan* out) {
    const int cols = (c->n_theta + C - 1) / C;
    int order[3] = {6, 4, 2};
    auto padded = [&](int cand) { return (cols + 32 * cand - 1) / (32 * cand) * (32 * cand); };
    std::stable_sort(order, order + 3, [&](int x, int y) { return padded(x) < padded(y); });   // ties keep the larger first
    for (int a = 0; a < 3; ++a)
        if (try_plan_cpl(c, acc16, C, want_ctas, order[a], out)) return true;
    return false;
}

// Pure host logic (no CUDA call): the smallest cluster of {1,2,4,8} CTAs whose layout fits, two CTAs per SM if possible.
bool choose_plan(const hough_ctx* c, Plan* best) {
    const bool acc16 = c->acc_dtype != HOUGH_ACC_U32;
    const int cands[5] = {1, 2, 4, 8, 16};   // 16 = non-portable cluster size, only when nothing smaller fits
    for (int ci = 0; ci < 5; ++ci) {
        const int C = cands[ci];
        if (c->opt_cluster && C != c->opt_cluster) continue;
        if (C > c->n_theta) continue;
        // prefer two CTAs per SM (phases of co-resident events overlap), else one
        const int first = (c->opt_ctas_per_sm == 1) ? 1 : 2;
        for (int want = first; want >= 1; --want)
            if (try_plan(c, acc16, C, want, best)) return true;
    }
    return false;
}

int make_plan(hough_ctx* c) {
    const bool acc16 = c->acc_dtype != HOUGH_ACC_U32;
    Plan best;
    if (!choose_plan(c, &best))
        return fail(HOUGH_ERR_UNSUPPORTED, "a %d x %d %s accumulator does not fit the shared memory of %s",
                    c->n_theta, c->n_rho, acc16 ? "u16" : "u32",
                    c->opt_cluster ? "the requested cluster size" : "a 16-CTA cluster");
    const void* fn = pick_kernel(best.acc16, best.csize > 1, best.cpl, false);
    int cur = -1;
    CUDA_TRY(cudaGetDevice(&cur));
    if (cur != c->device) return fail(HOUGH_ERR_INVALID_ARG, "the handle belongs to device %d but device %d is current", c->device, cur);
    if (int rc = prepare_kernel(c->device, fn, best.smem_bytes, best.csize)) return rc;
    int occ = 0;
    if (best.csize == 1) {
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, best.threads, best.smem_bytes));
        if (occ < 1) return fail(HOUGH_ERR_UNSUPPORTED, "kernel does not fit an SM (threads %d, smem %d)", best.threads, best.smem_bytes);
        if (occ > 2) occ = 2;
        best.ctas_per_sm = occ;
        best.grid_max = occ * c->sm_count;
    } else {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)(c->sm_count / best.csize * best.csize));
        cfg.blockDim = dim3((unsigned)best.threads);
        cfg.dynamicSmemBytes = (size_t)best.smem_bytes;
        cudaLaunchAttribute at{};
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = (unsigned)best.csize; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
        cfg.attrs = &at; cfg.numAttrs = 1;
        int ncl = 0;
        const cudaError_t oe = cudaOccupancyMaxActiveClusters(&ncl, fn, &cfg);
        if (oe != cudaSuccess) (void)cudaGetLastError();
        if (oe != cudaSuccess || ncl < 1)
            return fail(HOUGH_ERR_UNSUPPORTED, "no %d-CTA cluster of this kernel fits the device (%s)", best.csize,
                        oe != cudaSuccess ? cudaGetErrorString(oe) : "0 active clusters");
        best.grid_max = ncl * best.csize;
        best.ctas_per_sm = (best.grid_max + c->sm_count - 1) / c->sm_count;
    }
    c->plan = best;
    return HOUGH_OK;
}

int upload_table(hough_ctx* c, const float* h_cos, const float* h_sin) {
    float tmax = 0.0f, tmin_nz = INFINITY;
    for (int j = 0; j < c->n_theta; ++j) {
        if (!std::isfinite(h_cos[j]) || !std::isfinite(h_sin[j]))
            return fail(HOUGH_ERR_INVALID_ARG, "trig table entry %d is not finite", j);
        const float ac = std::fabs(h_cos[j]), as = std::fabs(h_sin[j]);
        tmax = std::fmax(tmax, std::fmax(ac, as));
        if (ac > 0.0f) tmin_nz = std::fmin(tmin_nz, ac);
        if (as > 0.0f) tmin_nz = std::fmin(tmin_nz, as);
    }
    CUDA_TRY(cudaMemcpy(c->d_cos, h_cos, sizeof(float) * c->n_theta, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(c->d_sin, h_sin, sizeof(float) * c->n_theta, cudaMemcpyHostToDevice));
    c->tmax = tmax;
    c->tmin_nz = tmin_nz;
    return HOUGH_OK;
}

float tame_bound(float inv, float rho_max, float tmax) {
    // hits with (|u|+|v|) * tmax <= 0.99 * (2^17/inv - rho_max) have |t| < 2^17 at every column
    double rho_lim = 131072.0 / (double)inv - (double)rho_max;
    if (!(rho_lim > 0.0)) return 0.0f;
    if (tmax <= 0.0f) return 3.0e38f;
    double b = 0.99 * rho_lim / (double)tmax;
    return b > 3.0e38 ? 3.0e38f : (float)b;
}

float ftz_min(float tmin_nz) {
    // |u| >= 2^-125 / tmin_nz  =>  |u * c_j| >= 2^-125 (before rounding) for every non-zero table entry:
    // the product is a normal number and the .ftz of the packed multiply never acts.  Never below 2^-125,
    // so that a subnormal u or v (flushed on input) is excluded too.
    if (!(tmin_nz > 0.0f) || !std::isfinite(tmin_nz)) return 2.3509887e-38f;   // all-zero table: nothing to flush
    double b = std::ldexp(1.0, -125) / (double)tmin_nz;
    if (b < std::ldexp(1.0, -125)) b = std::ldexp(1.0, -125);
    return b > 3.0e38 ? 3.0e38f : (float)(b * 1.0000002);
}

int launch(hough_ctx* c, const hough_io* io, cudaStream_t stream) {
    const Plan& pl = c->plan;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != c->device)   // tables and kernel attributes are per device
        return fail(HOUGH_ERR_INVALID_ARG, "the handle belongs to device %d but device %d is current", c->device, cur);
    KParams kp = pl.kp;
    kp.xy = (const float2*)io->d_xy;
    kp.off = io->d_event_offsets;
    kp.n_events = io->n_events;
    kp.keep = io->d_keep_mask;
    kp.peaks = io->d_peaks;
    kp.counts = io->d_counts;
    kp.kept_xy = (float2*)io->d_kept_xy;
    kp.kept_idx = io->d_kept_idx;
    kp.accum_dump = io->d_accum_dump;
    kp.cos_t = c->d_cos;
    kp.sin_t = c->d_sin;
    kp.n_theta = c->n_theta; kp.n_rho = c->n_rho; kp.threshold = c->threshold; kp.window = c->window;
    kp.max_peaks = c->max_peaks;
    kp.rho_max = c->rho_max; kp.inv = c->inv; kp.scale = (float)c->conformal_scale;
    kp.tame_bound = tame_bound(c->inv, c->rho_max, c->tmax);
    kp.ftz_min = ftz_min(c->tmin_nz);
    kp.force_slow = c->opt_vote_path == 1;
#ifdef HOUGH_DIAG
    kp.diag = c->opt_vote_path >= 2 ? c->opt_vote_path : 0;
#endif
    const bool ext = wants_ext(c);
    kp.peak_mode = c->peak_mode; kp.rel_permille = c->rel_permille; kp.nms_radius = c->nms_radius;
    kp.theta_wrap = c->theta_wrap; kp.keep_mode = c->keep_mode; kp.keep_tol = c->keep_tol;
    kp.stage_mode = c->stage_mode;
    kp.sched_mode = c->sched_mode;
    kp.select_mode = c->select_mode;
    if ((c->stage_mode == 1 || c->sched_mode == 1) && ((uintptr_t)io->d_xy & 15u) != 0)
        return fail(HOUGH_ERR_INVALID_ARG, "bulk-copy staging and the work-stealing scheduler need d_xy 16-byte aligned");
    if (c->sched_mode == 1 && (long long)io->n_events * pl.csize > 0x7FFFFFF0LL)
        return fail(HOUGH_ERR_UNSUPPORTED, "the work-stealing scheduler needs one CTA per event in one grid");
    const int C = pl.csize;
    // one CTA (cluster) per event: the hardware block scheduler deals events to the SM slots as they free up, which
    // balances events of different size; the kernel's event loop only matters beyond 2^31 CTAs
    long long want = (long long)io->n_events * C;
    int grid = (int)std::min<long long>(want, 0x7FFFFFF0LL);
    grid = grid / C * C;
    if (grid < C) grid = C;
    const void* fn = pick_kernel(pl.acc16, C > 1, pl.cpl, ext);
    if (ext)   // the extended instantiation is a different kernel: its attributes are set on first use (cheap afterwards)
        if (int rc = prepare_kernel(c->device, fn, pl.smem_bytes, C)) return rc;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)pl.threads);
    cfg.dynamicSmemBytes = (size_t)pl.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute at{};
    if (C > 1) {
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = (unsigned)C; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
        cfg.attrs = &at; cfg.numAttrs = 1;
    }
    void* args[1] = {(void*)&kp};
    CUDA_TRY(cudaLaunchKernelExC(&cfg, fn, args));
    c->launches.fetch_add(1);
    return HOUGH_OK;
}

}  // namespace

extern "C" {

hough_ctx* hough_create(int n_theta, int n_rho, float rho_max, int threshold, int window) {
    if (n_theta < 1 || n_theta > 65535 || n_rho < 1 || n_rho > 65535) {
        fail(HOUGH_ERR_INVALID_ARG, "n_theta and n_rho must be in 1..65535 (got %d, %d)", n_theta, n_rho);
        return nullptr;
    }
    if (!(rho_max > 0.0f) || !std::isfinite(rho_max)) { fail(HOUGH_ERR_INVALID_ARG, "rho_max must be finite and > 0"); return nullptr; }
    if (threshold < 1) { fail(HOUGH_ERR_INVALID_ARG, "threshold must be >= 1"); return nullptr; }
    if (window < 0 || window > 65535) { fail(HOUGH_ERR_INVALID_ARG, "window must be in 0..65535"); return nullptr; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        fail(HOUGH_ERR_CUDA, "no CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
        return nullptr;
    }
    hough_ctx* c = new (std::nothrow) hough_ctx();
    if (!c) { fail(HOUGH_ERR_NOMEM, "out of host memory"); return nullptr; }
    c->n_theta = n_theta; c->n_rho = n_rho; c->rho_max = rho_max; c->threshold = threshold; c->window = window;
    c->inv = (float)((double)n_rho / (2.0 * (double)rho_max));
    cudaDeviceProp prop;
    if (cudaGetDevice(&c->device) != cudaSuccess || cudaGetDeviceProperties(&prop, c->device) != cudaSuccess) {
        fail(HOUGH_ERR_CUDA, "cannot query the current CUDA device");
        delete c; return nullptr;
    }
    if (prop.major < 10) {
        fail(HOUGH_ERR_UNSUPPORTED, "built for sm_100a (B200); device is sm_%d%d", prop.major, prop.minor);
        delete c; return nullptr;
    }
    c->sm_count = prop.multiProcessorCount;
    c->smem_optin = (int)prop.sharedMemPerBlockOptin;
    if (cudaMalloc(&c->d_cos, sizeof(float) * n_theta) != cudaSuccess || cudaMalloc(&c->d_sin, sizeof(float) * n_theta) != cudaSuccess) {
        fail(HOUGH_ERR_NOMEM, "cudaMalloc of the trig table failed");
        hough_destroy(c); return nullptr;
    }
    std::vector<float> hc(n_theta), hs(n_theta);
    for (int j = 0; j < n_theta; ++j) {   // theta_j = j*pi/n_theta, left bin edges (reading Q3)
        double th = (double)j * M_PI / (double)n_theta;
        hc[j] = (float)std::cos(th);
        hs[j] = (float)std::sin(th);
    }
    if (upload_table(c, hc.data(), hs.data()) != HOUGH_OK || make_plan(c) != HOUGH_OK) { hough_destroy(c); return nullptr; }
    return c;
}

int hough_set_option(hough_ctx* c, int key, long long value) {
    if (!c) return fail(HOUGH_ERR_INVALID_ARG, "null handle");
    const int o_mp = c->max_peaks, o_acc = c->acc_dtype, o_sc = c->conformal_scale, o_cl = c->opt_cluster,
              o_cps = c->opt_ctas_per_sm, o_vp = c->opt_vote_path;
    switch (key) {   // options that need no new plan
        case HOUGH_OPT_PEAK_MODE:
            if (value != 0 && value != 1) return fail(HOUGH_ERR_INVALID_ARG, "peak mode must be 0 or 1");
            c->peak_mode = (int)value; return HOUGH_OK;
        case HOUGH_OPT_REL_THRESHOLD_PERMILLE:
            if (value < 0 || value > 1000) return fail(HOUGH_ERR_INVALID_ARG, "relative threshold must be 0..1000 permille");
            c->rel_permille = (int)value; return HOUGH_OK;
        case HOUGH_OPT_NMS_RADIUS:
            if (value < 0 || value > 64) return fail(HOUGH_ERR_INVALID_ARG, "NMS radius must be 0..64");
            c->nms_radius = (int)value; return HOUGH_OK;
        case HOUGH_OPT_THETA_WRAP:
            if (value != 0 && value != 1) return fail(HOUGH_ERR_INVALID_ARG, "theta wrap must be 0 or 1");
            c->theta_wrap = (int)value; return HOUGH_OK;
        case HOUGH_OPT_KEEP_MODE:
            if (value != 0 && value != 1) return fail(HOUGH_ERR_INVALID_ARG, "keep mode must be 0 or 1");
            c->keep_mode = (int)value; return HOUGH_OK;
        case HOUGH_OPT_STAGING:
            if (value != 0 && value != 1) return fail(HOUGH_ERR_INVALID_ARG, "staging must be 0 or 1");
            c->stage_mode = (int)value; return HOUGH_OK;
        case HOUGH_OPT_SCHEDULER:
            if (value != 0 && value != 1) return fail(HOUGH_ERR_INVALID_ARG, "scheduler must be 0 or 1");
            c->sched_mode = (int)value; return HOUGH_OK;
        case HOUGH_OPT_SELECT_MODE:
            if (value < 0 || value > 2) return fail(HOUGH_ERR_INVALID_ARG, "select mode must be 0, 1 or 2");
            c->select_mode = (int)value; return HOUGH_OK;
        default: break;
    }
    switch (key) {
        case HOUGH_OPT_MAX_PEAKS:
            if (value < 0 || value > 1048576) return fail(HOUGH_ERR_INVALID_ARG, "max_peaks must be in 0..1048576");
            c->max_peaks = (int)value; return HOUGH_OK;
        case HOUGH_OPT_ACC_DTYPE:
            if (value != HOUGH_ACC_AUTO && value != HOUGH_ACC_U16 && value != HOUGH_ACC_U32) return fail(HOUGH_ERR_INVALID_ARG, "bad accumulator dtype");
            c->acc_dtype = (int)value; break;
        case HOUGH_OPT_CONFORMAL_SCALE:
            if (value != 1 && value != 2) return fail(HOUGH_ERR_INVALID_ARG, "conformal scale must be 1 or 2");
            c->conformal_scale = (int)value; return HOUGH_OK;
        case HOUGH_OPT_CLUSTER_SIZE:
            if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8 && value != 16)
                return fail(HOUGH_ERR_INVALID_ARG, "cluster size must be 0,1,2,4,8,16");
            c->opt_cluster = (int)value; break;
        case HOUGH_OPT_CTAS_PER_SM:
            if (value < 0 || value > 2) return fail(HOUGH_ERR_INVALID_ARG, "ctas_per_sm must be 0,1,2");
            c->opt_ctas_per_sm = (int)value; break;
        case HOUGH_OPT_VOTE_PATH:
#ifdef HOUGH_DIAG   // bench-only build: 2 skips the voting loops, 3 skips everything after voting (outputs undefined)
            if (value < 0 || value > 3) return fail(HOUGH_ERR_INVALID_ARG, "vote path must be 0..3");
#else
            if (value < 0 || value > 1) return fail(HOUGH_ERR_INVALID_ARG, "vote path must be 0 or 1");
#endif
            c->opt_vote_path = (int)value; return HOUGH_OK;
        default:
            return fail(HOUGH_ERR_INVALID_ARG, "unknown option %d", key);
    }
    int rc = make_plan(c);
    if (rc != HOUGH_OK) {   // roll back: the handle stays usable with its previous configuration
        c->max_peaks = o_mp; c->acc_dtype = o_acc; c->conformal_scale = o_sc; c->opt_cluster = o_cl;
        c->opt_ctas_per_sm = o_cps; c->opt_vote_path = o_vp;
    }
    return rc;
}

int hough_set_option_f64(hough_ctx* c, int key, double value) {
    if (!c) return fail(HOUGH_ERR_INVALID_ARG, "null handle");
    switch (key) {
        case HOUGH_OPTF_KEEP_TOL:
            if (!(value >= 0.0)) return fail(HOUGH_ERR_INVALID_ARG, "the keep tolerance must be >= 0");
            c->keep_tol = value; return HOUGH_OK;
        case HOUGH_OPTF_B_FIELD_TESLA:
            if (!std::isfinite(value)) return fail(HOUGH_ERR_INVALID_ARG, "the field must be finite");
            c->b_field = value; return HOUGH_OK;
        default:
            return fail(HOUGH_ERR_INVALID_ARG, "unknown real-valued option %d", key);
    }
}

int hough_circles(hough_ctx* c, const float* d_xy, const int32_t* d_event_offsets, int n_events, const hough_peak* d_peaks,
                  const int32_t* d_counts, hough_circle* d_circles, hough_stream stream) {
    if (!c) return fail(HOUGH_ERR_INVALID_ARG, "null handle");
    if (n_events < 0) return fail(HOUGH_ERR_INVALID_ARG, "n_events < 0");
    if (n_events == 0 || c->max_peaks == 0) return HOUGH_OK;
    if (!d_xy || !d_event_offsets || !d_peaks || !d_counts || !d_circles) return fail(HOUGH_ERR_INVALID_ARG, "null device pointer");
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != c->device)
        return fail(HOUGH_ERR_INVALID_ARG, "the handle belongs to device %d but device %d is current", c->device, cur);
    hough::CParams cp{};
    cp.xy = (const float2*)d_xy; cp.off = d_event_offsets; cp.n_events = n_events; cp.peaks = d_peaks; cp.counts = d_counts;
    cp.out = d_circles; cp.cos_t = c->d_cos; cp.sin_t = c->d_sin;
    cp.n_theta = c->n_theta; cp.n_rho = c->n_rho; cp.window = c->window; cp.max_peaks = c->max_peaks;
    cp.rho_max = c->rho_max; cp.inv = c->inv; cp.scale = (float)c->conformal_scale; cp.b_field = c->b_field;
    const int grid = (int)std::min<long long>(n_events, 0x7FFFFFF0LL);
    void* args[1] = {(void*)&cp};
    CUDA_TRY(cudaLaunchKernel((const void*)&hough::hough_circles_kernel, dim3((unsigned)grid), dim3(256), args, 0, (cudaStream_t)stream));
    c->launches.fetch_add(1);
    return HOUGH_OK;
}

int hough_set_trig_table(hough_ctx* c, const float* h_cos, const float* h_sin) {
    if (!c || !h_cos || !h_sin) return fail(HOUGH_ERR_INVALID_ARG, "null argument");
    return upload_table(c, h_cos, h_sin);
}

long long hough_get_info(const hough_ctx* c, int key) {
    if (!c) return fail(HOUGH_ERR_INVALID_ARG, "null handle");
    switch (key) {
        case HOUGH_INFO_CLUSTER_SIZE: return c->plan.csize;
        case HOUGH_INFO_THREADS: return c->plan.threads;
        case HOUGH_INFO_SMEM_BYTES: return c->plan.smem_bytes;
        case HOUGH_INFO_CTAS_PER_SM: return c->plan.ctas_per_sm;
        case HOUGH_INFO_GRID_MAX: return c->plan.grid_max;
        case HOUGH_INFO_ACC_BITS: return c->plan.acc16 ? 16 : 32;
        case HOUGH_INFO_MAX_PEAKS: return c->max_peaks;
        case HOUGH_INFO_CHUNK_HITS: return c->plan.kp.chunk;
        case HOUGH_INFO_SM_COUNT: return c->sm_count;
        case HOUGH_INFO_LAUNCHES: return c->launches.load();
        default: return fail(HOUGH_ERR_INVALID_ARG, "unknown info key %d", key);
    }
}

int hough_run_ex(hough_ctx* c, const hough_io* io, hough_stream stream) {
    if (!c || !io) return fail(HOUGH_ERR_INVALID_ARG, "null handle or io");
    if (io->n_events < 0) return fail(HOUGH_ERR_INVALID_ARG, "n_events < 0");
    if (io->n_events == 0) return HOUGH_OK;
    if (!io->d_xy || !io->d_event_offsets || !io->d_keep_mask || !io->d_counts) return fail(HOUGH_ERR_INVALID_ARG, "null device pointer");
    if (!io->d_peaks && c->max_peaks > 0) return fail(HOUGH_ERR_INVALID_ARG, "d_peaks is null but max_peaks > 0");
    return launch(c, io, (cudaStream_t)stream);
}

int hough_run(hough_ctx* c, const float* d_xy, const int32_t* d_event_offsets, int n_events,
              uint8_t* d_keep_mask, hough_peak* d_peaks, int32_t* d_counts, hough_stream stream) {
    hough_io io{};
    io.d_xy = d_xy; io.d_event_offsets = d_event_offsets; io.n_events = n_events;
    io.d_keep_mask = d_keep_mask; io.d_peaks = d_peaks; io.d_counts = d_counts;
    return hough_run_ex(c, &io, stream);
}

int hough_run_host(hough_ctx* c, const float* h_xy, const int32_t* h_off, int n_events,
                   uint8_t* h_keep, hough_peak* h_peaks, int32_t* h_counts,
                   float* h_kept_xy, int32_t* h_kept_idx, hough_stream stream) {
    if (!c) return fail(HOUGH_ERR_INVALID_ARG, "null handle");
    if (n_events < 0) return fail(HOUGH_ERR_INVALID_ARG, "n_events < 0");
    if (n_events == 0) return HOUGH_OK;
    if (!h_off || !h_keep || !h_counts || (!h_peaks && c->max_peaks > 0)) return fail(HOUGH_ERR_INVALID_ARG, "null host pointer");
    // the hit arrays are indexed by the offsets themselves: a sub-batch passes the same h_xy / h_keep with h_off advanced
    const long long base = (long long)h_off[0], n_sub = (long long)h_off[n_events] - base;
    if (base < 0 || n_sub < 0 || (n_sub > 0 && !h_xy)) return fail(HOUGH_ERR_INVALID_ARG, "bad offsets or null h_xy");
    cudaStream_t st = (cudaStream_t)stream;
    const long long n_peaks_cap = (long long)n_events * c->max_peaks;

    // one staging area per stream (N4c: streams + pinned memory + asynchronous transfers): calls on
    // different streams overlap their H2D copy, kernel and D2H copies
    Staging* sg = nullptr;
    {
        std::lock_guard<std::mutex> lk(c->staging_mu);
        for (auto& x : c->staging) if (x.used && x.stream == st) sg = &x;
        if (!sg) for (auto& x : c->staging) if (!x.used) { sg = &x; break; }
        if (!sg) {                                    // all slots taken: recycle the least recently used one
            sg = &c->staging[0];
            for (auto& x : c->staging) if (x.tick < sg->tick) sg = &x;
            CUDA_TRY(cudaStreamSynchronize(sg->stream));
        }
        sg->used = true; sg->stream = st; sg->tick = ++c->staging_tick;
    }
    if (n_sub + 1 > sg->cap_hits || n_events > sg->cap_events || n_peaks_cap > sg->cap_peaks) {
        CUDA_TRY(cudaStreamSynchronize(st));          // the slot's earlier work runs on this very stream
        sg->release();
        sg->cap_hits = n_sub + 17; sg->cap_events = n_events; sg->cap_peaks = n_peaks_cap + 1;
        cudaError_t e1 = cudaMalloc(&sg->xy, sizeof(float) * 2 * sg->cap_hits);
        cudaError_t e2 = cudaMalloc(&sg->off, sizeof(int32_t) * ((size_t)sg->cap_events + 1));
        cudaError_t e3 = cudaMalloc(&sg->keep, (size_t)sg->cap_hits);
        cudaError_t e4 = cudaMalloc(&sg->peaks, sizeof(hough_peak) * (size_t)sg->cap_peaks);
        cudaError_t e5 = cudaMalloc(&sg->counts, sizeof(int32_t) * 2 * (size_t)sg->cap_events);
        cudaError_t e6 = cudaMalloc(&sg->kept_xy, sizeof(float) * 2 * sg->cap_hits);
        cudaError_t e7 = cudaMalloc(&sg->kept_idx, sizeof(int32_t) * sg->cap_hits);
        if (e1 || e2 || e3 || e4 || e5 || e6 || e7) {
            sg->release();
            return fail(HOUGH_ERR_NOMEM, "cudaMalloc of the staging area failed");
        }
    }
    // the kernel leaves peak entries past n_stored and kept entries past n_kept untouched: zero what goes back
    if (c->max_peaks > 0) CUDA_TRY(cudaMemsetAsync(sg->peaks, 0, sizeof(hough_peak) * (size_t)n_peaks_cap, st));
    if (h_kept_xy && n_sub > 0) CUDA_TRY(cudaMemsetAsync(sg->kept_xy, 0, sizeof(float) * 2 * n_sub, st));
    if (h_kept_idx && n_sub > 0) CUDA_TRY(cudaMemsetAsync(sg->kept_idx, 0, sizeof(int32_t) * n_sub, st));
    // hits keep the parity of their absolute index in the staging buffer (hit `base` goes to slot base & 1), so that the
    // pointer handed to the kernel stays 16-byte aligned (bulk-copy staging relies on it)
    const long long par = base & 1;
    if (n_sub > 0) CUDA_TRY(cudaMemcpyAsync(sg->xy + 2 * par, h_xy + 2 * base, sizeof(float) * 2 * n_sub, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(sg->off, h_off, sizeof(int32_t) * ((size_t)n_events + 1), cudaMemcpyHostToDevice, st));
    // The staged hit arrays hold hits base .. base+n_sub-1 at positions 0 ..; the kernel indexes them by the (absolute)
    // offsets, so it is handed pointers moved back by `base` -- dereferenced only at base and beyond.
    hough_io io{};
    io.d_xy = sg->xy + 2 * par - 2 * base; io.d_event_offsets = sg->off; io.n_events = n_events;
    io.d_keep_mask = sg->keep - base; io.d_peaks = sg->peaks; io.d_counts = sg->counts;
    io.d_kept_xy = h_kept_xy ? sg->kept_xy - 2 * base : nullptr;
    io.d_kept_idx = h_kept_idx ? sg->kept_idx - base : nullptr;
    int rc = launch(c, &io, st);
    if (rc != HOUGH_OK) return rc;
    if (n_sub > 0) CUDA_TRY(cudaMemcpyAsync(h_keep + base, sg->keep, (size_t)n_sub, cudaMemcpyDeviceToHost, st));
    if (c->max_peaks > 0) CUDA_TRY(cudaMemcpyAsync(h_peaks, sg->peaks, sizeof(hough_peak) * (size_t)n_peaks_cap, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(h_counts, sg->counts, sizeof(int32_t) * 2 * (size_t)n_events, cudaMemcpyDeviceToHost, st));
    if (h_kept_xy && n_sub > 0) CUDA_TRY(cudaMemcpyAsync(h_kept_xy + 2 * base, sg->kept_xy, sizeof(float) * 2 * n_sub, cudaMemcpyDeviceToHost, st));
    if (h_kept_idx && n_sub > 0) CUDA_TRY(cudaMemcpyAsync(h_kept_idx + base, sg->kept_idx, sizeof(int32_t) * n_sub, cudaMemcpyDeviceToHost, st));
    return HOUGH_OK;
}

void hough_destroy(hough_ctx* c) {
    if (!c) return;
    cudaFree(c->d_cos); cudaFree(c->d_sin);
    for (auto& x : c->staging) x.release();
    delete c;
}

const char* hough_strerror(int status) {
    switch (status) {
        case HOUGH_OK: return "ok";
        case HOUGH_ERR_INVALID_ARG: return "invalid argument";
        case HOUGH_ERR_UNSUPPORTED: return "unsupported configuration";
        case HOUGH_ERR_CUDA: return "CUDA error";
        case HOUGH_ERR_NOMEM: return "out of memory";
        default: return "unknown status";
    }
}

const char* hough_last_error(void) { return g_err; }

int hough_plan_describe(int n_theta, int n_rho, int acc_dtype, int cluster_size, int ctas_per_sm, int smem_optin,
                        long long* out, int n_out) {
    if (n_theta < 1 || n_theta > 65535 || n_rho < 1 || n_rho > 65535 || !out || n_out < HOUGH_PLAN_N_FIELDS)
        return fail(HOUGH_ERR_INVALID_ARG, "bad argument");
    if (acc_dtype != HOUGH_ACC_AUTO && acc_dtype != HOUGH_ACC_U16 && acc_dtype != HOUGH_ACC_U32) return fail(HOUGH_ERR_INVALID_ARG, "bad accumulator dtype");
    if (cluster_size != 0 && cluster_size != 1 && cluster_size != 2 && cluster_size != 4 && cluster_size != 8 && cluster_size != 16)
        return fail(HOUGH_ERR_INVALID_ARG, "cluster size must be 0,1,2,4,8,16");
    if (ctas_per_sm < 0 || ctas_per_sm > 2) return fail(HOUGH_ERR_INVALID_ARG, "ctas_per_sm must be 0,1,2");
    hough_ctx c;
    c.n_theta = n_theta; c.n_rho = n_rho; c.threshold = 1; c.window = 0; c.rho_max = 1.0f; c.inv = 1.0f;
    c.acc_dtype = acc_dtype; c.opt_cluster = cluster_size; c.opt_ctas_per_sm = ctas_per_sm;
    c.smem_optin = smem_optin > 0 ? smem_optin : 232448;   // B200: 227 KB per CTA with opt-in
    Plan pl;
    if (!choose_plan(&c, &pl)) return fail(HOUGH_ERR_UNSUPPORTED, "the accumulator does not fit");
    const KParams& k = pl.kp;
    const long long v[HOUGH_PLAN_N_FIELDS] = {
        pl.csize, pl.threads, pl.smem_bytes, pl.acc16 ? 16 : 32, pl.cpl, k.cols_per_cta, k.n_groups, k.n_stripes,
        k.pitch_b, k.wpr, k.chunk, k.region_bytes, k.pbm_off, k.pbm_bytes, k.hb_off, k.misc_off,
        k.w8_off, k.w8_pitch, k.mcf_off, k.msf_off, k.colq_off, k.stash_off, k.cnt_off, k.gcnt_off, k.rcp_groups, k.rcp_2s, k.circ_cap};
    for (int i = 0; i < HOUGH_PLAN_N_FIELDS; ++i) out[i] = v[i];
    return HOUGH_OK;
}

int hough_debug_tame_bounds(int n_rho, float rho_max, float table_max, float table_min_nz, float* out2) {
    if (n_rho < 1 || !(rho_max > 0.0f) || !out2) return fail(HOUGH_ERR_INVALID_ARG, "bad argument");
    const float inv = (float)((double)n_rho / (2.0 * (double)rho_max));
    out2[0] = tame_bound(inv, rho_max, table_max);
    out2[1] = ftz_min(table_min_nz);
    return HOUGH_OK;
}

int hough_debug_bounds_enabled(void) {
#ifdef HOUGH_DEBUG_BOUNDS
    return 1;
#else
    return 0;
#endif
}

const char* hough_version(void) {
#ifdef HOUGH_DEBUG_BOUNDS
    return "hough-b200 0.2 (sm_100a, debug bounds)";
#else
    return "hough-b200 0.2 (sm_100a)";
#endif
}

}  // extern "C"
