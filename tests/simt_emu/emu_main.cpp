// emu_main.cpp -- TEST INFRASTRUCTURE.  Runs paper_2607_04067_b200/csrc/hough_kernel.cuh on the CPU under the SIMT
// shim (simt_shim.h): `hough_emu <in.bin> <out.bin>`.  The launch shape and shared-memory layout come from the
// product's own planner (hough_plan_describe / hough_debug_tame_bounds, passed in by the Python side), so what runs
// here is the kernel exactly as hough_run would launch it, one cluster after the other.  Every global buffer and
// every CTA's shared memory ends at an inaccessible page: an out-of-bounds access is a crash, not a wrong number.
#include "simt_shim.h"

#ifndef HOUGH_HOST_EMU
#error "build with -DHOUGH_HOST_EMU (tests/simt_emu/__init__.py)"
#endif
#ifdef HOUGH_KERNEL_HEADER      // the mutation tests compile a modified copy of the kernel (tests/test_kernel_races.py)
#include HOUGH_KERNEL_HEADER
#else
#include "../../paper_2607_04067_b200/csrc/hough_kernel.cuh"
#endif

namespace {

hough::KParams kp;
int g_acc16, g_cl, g_cpl;

int g_ext;
hough::CParams cpar;

template <bool ACC16, bool CL, bool EXT>
void call_cpl() {
    switch (g_cpl) {
        case 6: hough::hough_event_kernel<ACC16, CL, 6, EXT>(kp); break;
        case 4: hough::hough_event_kernel<ACC16, CL, 4, EXT>(kp); break;
        default: hough::hough_event_kernel<ACC16, CL, 2, EXT>(kp); break;
    }
}

template <bool EXT>
void entry_t() {
    if (g_acc16) { if (g_cl) call_cpl<true, true, EXT>(); else call_cpl<true, false, EXT>(); }
    else { if (g_cl) call_cpl<false, true, EXT>(); else call_cpl<false, false, EXT>(); }
}

void entry() { if (g_ext) entry_t<true>(); else entry_t<false>(); }   // the same choice hough_api.cu's pick_kernel makes
void entry_circles() { hough::hough_circles_kernel(cpar); }

template <class T> void rd(FILE* f, T* p, size_t n) {
    if (n && fread(p, sizeof(T), n, f) != n) emu::die("short input file");
}

}  // namespace

int main(int argc, char** argv) {
    if (argc != 3) emu::die("usage: hough_emu in.bin out.bin");
    FILE* f = fopen(argv[1], "rb");
    if (!f) emu::die("cannot open the input file");
    // header: 24 ints, 27 plan fields (int32), 5 floats, 2 doubles
    int h[24];
    int plan[27];
    float fl[5];
    double dbl[2];
    rd(f, h, 24); rd(f, plan, 27); rd(f, fl, 5); rd(f, dbl, 2);
    const int n_theta = h[0], n_rho = h[1], threshold = h[2], window = h[3], max_peaks = h[4];
    g_acc16 = h[5]; g_cl = h[6]; g_cpl = h[7];
    const int csize = h[8], threads = h[9], smem_bytes = h[10], force_slow = h[11], n_events = h[12], n_total = h[13];
    const int want_kept = h[14], want_accum = h[15], grid_clusters = h[16];
    const int peak_mode = h[17], rel_permille = h[18], nms_radius = h[19], theta_wrap = h[20], keep_mode = h[21], want_circles = h[22], stage_mode = h[23] & 1, sched_mode = (h[23] >> 1) & 1, select_mode = (h[23] >> 2) & 3;
    g_ext = peak_mode != 0 || theta_wrap != 0 || keep_mode != 0 || stage_mode != 0 || sched_mode != 0 || select_mode != 0;
    std::vector<float> cos_t(n_theta), sin_t(n_theta);
    rd(f, cos_t.data(), n_theta); rd(f, sin_t.data(), n_theta);
    emu::Guarded b_off, b_xy, b_keep, b_peaks, b_counts, b_kxy, b_kidx, b_acc;
    b_off.alloc(4 * (size_t)(n_events + 1));
    // d_xy is 16-byte aligned (the promise bulk-copy staging relies on); it ends at the guard page when n_total is even,
    // one hit before it when odd (emu::bulk_check then catches a copy that reads past the batch's last hit)
    b_xy.alloc(8 * (size_t)n_total + 16);
    unsigned char* xy_base = b_xy.ptr + ((n_total & 1) ? 8 : 16);
    emu::bulk_lo = xy_base; emu::bulk_hi = xy_base + 8 * (size_t)n_total;
    rd(f, (int*)b_off.ptr, n_events + 1);
    rd(f, (float*)xy_base, 2 * (size_t)n_total);
    fclose(f);
    const size_t peaks_bytes = 8 * (size_t)n_events * max_peaks, accum_bytes = 4 * (size_t)n_events * n_theta * n_rho;
    b_keep.alloc((size_t)n_total + 1); b_peaks.alloc(peaks_bytes + 8); b_counts.alloc(8 * (size_t)n_events);
    b_kxy.alloc(8 * (size_t)n_total + 8); b_kidx.alloc(4 * (size_t)n_total + 4); b_acc.alloc(accum_bytes + 4);
    memset(b_keep.ptr, 7, b_keep.bytes);
    memset(b_peaks.ptr, 0xFF, b_peaks.bytes);
    for (int i = 0; i < 2 * n_events; ++i) ((int*)b_counts.ptr)[i] = -99;
    memset(b_kxy.ptr, 0, b_kxy.bytes);
    for (int i = 0; i <= n_total; ++i) ((int*)b_kidx.ptr)[i] = -5;
    memset(b_acc.ptr, 0xEE, b_acc.bytes);
#ifdef EMU_RACE                  // race check: the output buffers (the inputs are only ever read)
    emu::race::track(b_keep.ptr, b_keep.bytes, false, -1, "keep");
    emu::race::track(b_peaks.ptr, b_peaks.bytes, false, -1, "peaks");
    emu::race::track(b_counts.ptr, b_counts.bytes, false, -1, "counts");
    emu::race::track(b_kxy.ptr, b_kxy.bytes, false, -1, "kept_xy");
    emu::race::track(b_kidx.ptr, b_kidx.bytes, false, -1, "kept_idx");
    if (want_accum) emu::race::track(b_acc.ptr, b_acc.bytes, false, -1, "accum_dump");
#endif

    kp = hough::KParams();
    // the buffers END at a guard page; an empty buffer still gets a valid pointer (one spare element in front)
    kp.xy = (const float2*)xy_base;
    kp.off = (const int*)b_off.ptr;
    kp.n_events = n_events;
    kp.keep = b_keep.ptr + 1;
    kp.peaks = (hough_peak*)(b_peaks.ptr + 8);
    kp.counts = (int*)b_counts.ptr;
    kp.kept_xy = want_kept ? (float2*)(b_kxy.ptr + 8) : nullptr;
    kp.kept_idx = want_kept ? (int*)(b_kidx.ptr + 4) : nullptr;
    kp.accum_dump = want_accum ? (unsigned*)(b_acc.ptr + 4) : nullptr;
    kp.cos_t = cos_t.data(); kp.sin_t = sin_t.data();
    kp.n_theta = n_theta; kp.n_rho = n_rho; kp.threshold = threshold; kp.window = window; kp.max_peaks = max_peaks;
    kp.rho_max = fl[0]; kp.inv = fl[1]; kp.scale = fl[2]; kp.tame_bound = fl[3]; kp.ftz_min = fl[4];
    kp.force_slow = force_slow;
    kp.csize = csize;
    // plan fields in the order of enum hough_plan_field (include/hough_debug.h)
    kp.cols_per_cta = plan[5]; kp.n_groups = plan[6]; kp.n_stripes = plan[7]; kp.pitch_b = plan[8]; kp.wpr = plan[9];
    kp.chunk = plan[10]; kp.region_bytes = plan[11]; kp.pbm_off = plan[12]; kp.pbm_bytes = plan[13]; kp.hb_off = plan[14];
    kp.misc_off = plan[15]; kp.w8_off = plan[16]; kp.w8_pitch = plan[17]; kp.mcf_off = plan[18]; kp.msf_off = plan[19];
    kp.colq_off = plan[20]; kp.stash_off = plan[21]; kp.cnt_off = plan[22]; kp.gcnt_off = plan[23];
    kp.rcp_groups = (unsigned)plan[24]; kp.rcp_2s = (unsigned)plan[25]; kp.circ_cap = plan[26];
    kp.peak_mode = peak_mode; kp.rel_permille = rel_permille; kp.nms_radius = nms_radius; kp.theta_wrap = theta_wrap;
    kp.keep_mode = keep_mode; kp.keep_tol = dbl[0]; kp.stage_mode = stage_mode; kp.sched_mode = sched_mode; kp.select_mode = select_mode;
    kp.vpr = kp.pitch_b / 16;
    if (plan[0] != csize || plan[1] != threads || plan[2] != smem_bytes || plan[4] != g_cpl || (plan[3] == 16) != (g_acc16 != 0))
        emu::die("header and plan disagree");

    // hough_run launches one cluster per event; a smaller grid also exercises the kernel's event loop
    const int n_clusters = grid_clusters > 0 ? (grid_clusters < n_events ? grid_clusters : n_events) : n_events;
    // (with scheduler mode 1 a running CTA takes not-yet-launched CTAs out of the grid: emu::next_unlaunched)
    emu::next_unlaunched = 0;
    while (emu::next_unlaunched < n_clusters) {
        const int c = emu::next_unlaunched++;
        emu::g.n_clusters_ = n_clusters;
        emu::run_cluster(c, n_clusters, csize, threads, (size_t)smem_bytes, entry);
    }

    // N1: hough_circles on the peaks just written (grid = one 256-thread CTA per event, as hough_api.cu launches it)
    emu::Guarded b_circ;
    const size_t circ_bytes = sizeof(hough_circle) * (size_t)n_events * max_peaks;
    b_circ.alloc(circ_bytes + sizeof(hough_circle));
    memset(b_circ.ptr, 0xFF, b_circ.bytes);
    if (want_circles && max_peaks > 0) {
#ifdef EMU_RACE
        emu::race::new_launch();
        emu::race::track(b_circ.ptr, b_circ.bytes, false, -1, "circles");
#endif
        cpar = hough::CParams();
        cpar.xy = kp.xy; cpar.off = kp.off; cpar.n_events = n_events; cpar.peaks = kp.peaks; cpar.counts = kp.counts;
        cpar.out = (hough_circle*)(b_circ.ptr + sizeof(hough_circle)); cpar.cos_t = kp.cos_t; cpar.sin_t = kp.sin_t;
        cpar.n_theta = n_theta; cpar.n_rho = n_rho; cpar.window = window; cpar.max_peaks = max_peaks;
        cpar.rho_max = kp.rho_max; cpar.inv = kp.inv; cpar.scale = kp.scale; cpar.b_field = dbl[1];
        const int cgrid = grid_clusters > 0 ? (grid_clusters < n_events ? grid_clusters : n_events) : n_events;
        for (int c = 0; c < cgrid; ++c) emu::run_cluster(c, cgrid, 1, 256, 16, entry_circles);
    }

    FILE* o = fopen(argv[2], "wb");
    if (!o) emu::die("cannot open the output file");
    fwrite(b_keep.ptr + 1, 1, (size_t)n_total, o);
    fwrite(b_peaks.ptr + 8, 1, peaks_bytes, o);
    fwrite(b_counts.ptr, 4, 2 * (size_t)n_events, o);
    fwrite(b_kxy.ptr + 8, 4, 2 * (size_t)n_total, o);
    fwrite(b_kidx.ptr + 4, 4, (size_t)n_total, o);
    if (want_accum) fwrite(b_acc.ptr + 4, 1, accum_bytes, o);
    if (want_circles) fwrite(b_circ.ptr + sizeof(hough_circle), 1, circ_bytes, o);
    fclose(o);
#ifdef EMU_RACE
    for (auto& kv : emu::race::profile)
        fprintf(stderr, "PROF pc 0x%llx %s %s %llu\n", kv.first >> 8, (kv.first & 16) ? "shared" : "global",
                (const char*[]){"none", "read", "write", "atomic", "async"}[kv.first & 7], kv.second);
    if (emu::race::n_reports) { fprintf(stderr, "%lu race report(s)\n", emu::race::n_reports); return 66; }
#endif
    return 0;
}
