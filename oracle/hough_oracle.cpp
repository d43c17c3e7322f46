// hough_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU restatement of the conformal-mapped,
// matrix-form Hough transform of arxiv/paper_2607_04067, one event
// at a time, step by step in the paper's order.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call this file.  It shares no code with
// paper_2607_04067_b200/ (the CUDA path) and includes none of its headers.
//
// Build (see oracle/build.py):
//   g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC -pthread
// -ffp-contract=off forbids FMA contraction, so every fp32 operation below
// rounds once, to nearest-even, exactly as written (reading Q12).
//
// Steps and the passages they restate (SURVEY.md section 8(c) readings Q1..Q12
// are listed in DESIGN.md):
//   S1 conformal map        PAPER.md:52-57  Eq. (1)
//   S2 rho row + bin + vote PAPER.md:69 (rho = u cos + v sin), :73 (equal-width
//                           bins), :92-100 (matrix R, column accumulation)
//   S3 threshold + local max PAPER.md:75 (threshold, NMS in the neighbourhood)
//   S4 peak list            PAPER.md:75, :106 (only peaks are returned)
//   S5 hit selection        PAPER.md:44, :75 (filter hits by the candidates)
//   S6 compaction           PAPER.md:118-123 (N_select of Eq. (8))
//
// Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"): P1 closed form of a
// circle through the origin, P2 vote-sum invariant, P3 hand-worked example W1
// (tests/golden/w1_*.txt), P4 permutation invariance, P5 exact rescaling,
// P6 fp64 cross-check, P7 monotonicity.  Parity unpinned: none of S1..S6.
// (The paper's physics tables R_c, R_s etc. need its datasets: out of scope.)

#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

struct Params {
    int n_theta;
    int n_rho;
    float rho_max;     // fp32, same units as 1/hit-coordinates
    float inv;         // (float)((double)n_rho / (2.0 * (double)rho_max))
    int threshold;     // absolute vote count (reading Q7)
    int window;        // keep window half-width w, in bins (reading Q10)
    int max_peaks;     // peaks stored per event; n_peaks counts all
    float scale;       // conformal scale 1 or 2 (reading Q1)
    int acc_u16;       // 1: events with > 65535 hits yield {-1,-1}
    const float* cos_t;  // [n_theta] fp32 table, passed in as data (Q3)
    const float* sin_t;  // [n_theta]
};

// S1. Eq. (1):  u = x/(x^2+y^2), v = y/(x^2+y^2), times `scale`
// (scale = 1 is the equation as printed; 2 is the variant Eq. (2) implies).
inline void conformal(float x, float y, float scale, float* u, float* v) {
    float xx = x * x;
    float yy = y * y;
    float d = xx + yy;
    float u1 = x / d;
    float v1 = y / d;
    *u = scale * u1;   // exact for scale in {1,2}
    *v = scale * v1;
}

// S2 (one cell).  rho = u cos(theta_j) + v sin(theta_j)
// t = (rho + rho_max) * inv ; bin k = floor(t) if 0 <= t < n_rho, else the
// vote is dropped (readings Q4, Q5).  Returns k, or -1 when dropped.
inline int rho_bin(float u, float v, float c, float s, const Params& p) {
    float uc = u * c;
    float vs = v * s;
    float rho = uc + vs;
    float shifted = rho + p.rho_max;
    float t = shifted * p.inv;
    if (t >= 0.0f && t < (float)p.n_rho) return (int)t;
    return -1;   // also taken for NaN
}

// S2 (whole event).  A is [n_theta][n_rho], theta-major (reading Q6), zeroed here.
void accumulate(const float* xy, int n_hits, const Params& p, uint32_t* A) {
    std::memset(A, 0, sizeof(uint32_t) * (size_t)p.n_theta * (size_t)p.n_rho);
    for (int i = 0; i < n_hits; ++i) {
        float u, v;
        conformal(xy[2 * i], xy[2 * i + 1], p.scale, &u, &v);
        for (int j = 0; j < p.n_theta; ++j) {
            int k = rho_bin(u, v, p.cos_t[j], p.sin_t[j], p);
            if (k >= 0) A[(size_t)j * p.n_rho + k] += 1u;
        }
    }
}

inline uint32_t cell(const uint32_t* A, const Params& p, int j, int k) {
    if (j < 0 || j >= p.n_theta || k < 0 || k >= p.n_rho) return 0u;  // outside = 0, no theta wrap (Q8)
    return A[(size_t)j * p.n_rho + k];
}

// S3 + S4.  Raster order (j major, then k).  A cell is a peak iff a >= thr,
// a > every 3x3 neighbour that precedes it in raster order and a >= every one
// that follows (reading Q8).  peaks_out holds (j, k, votes) triples for the
// first max_peaks peaks; the return value counts all of them.
int find_peaks(const uint32_t* A, const Params& p, uint32_t* peaks_out /* [max_peaks][3] */) {
    int n_peaks = 0;
    for (int j = 0; j < p.n_theta; ++j) {
        for (int k = 0; k < p.n_rho; ++k) {
            uint32_t a = cell(A, p, j, k);
            if (a < (uint32_t)p.threshold) continue;
            bool is_peak = true;
            for (int dj = -1; dj <= 1 && is_peak; ++dj) {
                for (int dk = -1; dk <= 1; ++dk) {
                    if (dj == 0 && dk == 0) continue;
                    uint32_t n = cell(A, p, j + dj, k + dk);
                    bool precedes = (dj < 0) || (dj == 0 && dk < 0);
                    if (precedes ? !(a > n) : !(a >= n)) { is_peak = false; break; }
                }
            }
            if (!is_peak) continue;
            if (n_peaks < p.max_peaks) {
                peaks_out[3 * n_peaks + 0] = (uint32_t)j;
                peaks_out[3 * n_peaks + 1] = (uint32_t)k;
                peaks_out[3 * n_peaks + 2] = a;
            }
            ++n_peaks;
        }
    }
    return n_peaks;
}

// S5.  keep_i = 1 iff some STORED peak (j_p,k_p) and some column
// j in [j_p-w, j_p+w] (clipped to the array) has a valid bin(i,j) with
// |bin(i,j) - k_p| <= w  (reading Q10).
void select_hits(const float* xy, int n_hits, const Params& p,
                 const uint32_t* peaks, int n_stored, uint8_t* keep) {
    for (int i = 0; i < n_hits; ++i) {
        float u, v;
        conformal(xy[2 * i], xy[2 * i + 1], p.scale, &u, &v);
        uint8_t kp = 0;
        for (int q = 0; q < n_stored && !kp; ++q) {
            int jp = (int)peaks[3 * q + 0];
            int kpk = (int)peaks[3 * q + 1];
            int jlo = jp - p.window; if (jlo < 0) jlo = 0;
            int jhi = jp + p.window; if (jhi > p.n_theta - 1) jhi = p.n_theta - 1;
            for (int j = jlo; j <= jhi; ++j) {
                int k = rho_bin(u, v, p.cos_t[j], p.sin_t[j], p);
                if (k < 0) continue;
                int dk = k - kpk; if (dk < 0) dk = -dk;
                if (dk <= p.window) { kp = 1; break; }
            }
        }
        keep[i] = kp;
    }
}

// One event, S1..S6.  Outputs are written at the event's own offset `off`
// (reading Q11).  accum_out may be null.
void run_event(const float* xy_all, int off, int n_hits, const Params& p,
               uint8_t* keep_all, uint32_t* peaks_ev /* [max_peaks][3] */, int32_t* counts_ev /* [2] */,
               float* kept_xy_all, int32_t* kept_idx_all, uint32_t* accum_out,
               std::vector<uint32_t>& scratch) {
    if (p.acc_u16 && n_hits > 65535) {   // a u16 cell could wrap: refuse the event
        counts_ev[0] = -1; counts_ev[1] = -1;
        return;
    }
    const float* xy = xy_all + 2 * (size_t)off;
    uint32_t* A = accum_out;
    if (!A) {
        scratch.resize((size_t)p.n_theta * p.n_rho);
        A = scratch.data();
    }
    accumulate(xy, n_hits, p, A);
    int n_peaks = find_peaks(A, p, peaks_ev);
    int n_stored = n_peaks < p.max_peaks ? n_peaks : p.max_peaks;
    uint8_t* keep = keep_all + off;
    select_hits(xy, n_hits, p, peaks_ev, n_stored, keep);
    // S6: stable compaction in original order.
    int m = 0;
    for (int i = 0; i < n_hits; ++i) {
        if (keep[i]) {
            if (kept_xy_all) {
                kept_xy_all[2 * (size_t)(off + m) + 0] = xy[2 * i + 0];
                kept_xy_all[2 * (size_t)(off + m) + 1] = xy[2 * i + 1];
            }
            if (kept_idx_all) kept_idx_all[off + m] = i;
            ++m;
        }
    }
    counts_ev[0] = n_peaks;
    counts_ev[1] = m;
}

}  // namespace

extern "C" {

// Flat argument list so that ctypes can call it without a struct mirror.
// xy [n_total][2] fp32; offsets [n_events+1] int32 (CSR); keep [n_total] u8;
// peaks [n_events][max_peaks][3] u32 (theta_bin, rho_bin, votes);
// counts [n_events][2] int32 {n_peaks (untruncated), n_kept};
// kept_xy [n_total][2], kept_idx [n_total], accum [n_events][n_theta][n_rho] u32
// may be null.  n_threads <= 1: plain loop over events on the calling thread;
// n_threads > 1: the same per-event function over contiguous event ranges,
// one std::thread each (events are independent).
// Returns 0, or -1 on a bad argument.
int oracle_run(const float* xy, const int32_t* offsets, int n_events,
               int n_theta, int n_rho, float rho_max, int threshold, int window,
               int max_peaks, int conformal_scale, int acc_u16,
               const float* cos_t, const float* sin_t,
               uint8_t* keep, uint32_t* peaks, int32_t* counts,
               float* kept_xy, int32_t* kept_idx, uint32_t* accum, int n_threads) {
    if (n_theta < 1 || n_rho < 1 || !(rho_max > 0.0f) || threshold < 1 || window < 0 || max_peaks < 0) return -1;
    if (conformal_scale != 1 && conformal_scale != 2) return -1;
    if (n_events < 0) return -1;
    Params p;
    p.n_theta = n_theta; p.n_rho = n_rho; p.rho_max = rho_max;
    p.inv = (float)((double)n_rho / (2.0 * (double)rho_max));
    p.threshold = threshold; p.window = window; p.max_peaks = max_peaks;
    p.scale = (float)conformal_scale; p.acc_u16 = acc_u16;
    p.cos_t = cos_t; p.sin_t = sin_t;

    auto range = [&](int e0, int e1) {
        std::vector<uint32_t> scratch;
        for (int e = e0; e < e1; ++e) {
            int off = offsets[e];
            int n = offsets[e + 1] - off;
            run_event(xy, off, n, p, keep, peaks + (size_t)e * max_peaks * 3, counts + 2 * (size_t)e,
                      kept_xy, kept_idx,
                      accum ? accum + (size_t)e * n_theta * n_rho : nullptr, scratch);
        }
    };
    if (n_threads <= 1 || n_events <= 1) {
        range(0, n_events);
    } else {
        if (n_threads > n_events) n_threads = n_events;
        std::vector<std::thread> pool;
        for (int t = 0; t < n_threads; ++t) {
            int e0 = (int)((long long)n_events * t / n_threads);
            int e1 = (int)((long long)n_events * (t + 1) / n_threads);
            pool.emplace_back(range, e0, e1);
        }
        for (auto& th : pool) th.join();
    }
    return 0;
}

// Single-cell helpers exposed for the pins (so a test can probe S1 and S2
// without running an event).
void oracle_conformal(float x, float y, int conformal_scale, float* u, float* v) {
    conformal(x, y, (float)conformal_scale, u, v);
}

int oracle_rho_bin(float u, float v, float c, float s, float rho_max, int n_rho) {
    Params p{};
    p.n_rho = n_rho; p.rho_max = rho_max;
    p.inv = (float)((double)n_rho / (2.0 * (double)rho_max));
    return rho_bin(u, v, c, s, p);
}

// S3 + S4 alone, on a caller-made accumulator A [n_theta][n_rho] (so that a pin can hand-craft plateaus and borders
// and check find_peaks itself).  Returns n_peaks (untruncated); peaks_out [max_peaks][3].
int oracle_find_peaks(const uint32_t* A, int n_theta, int n_rho, int threshold, int max_peaks, uint32_t* peaks_out) {
    Params p{};
    p.n_theta = n_theta; p.n_rho = n_rho; p.threshold = threshold; p.max_peaks = max_peaks;
    return find_peaks(A, p, peaks_out);
}

}  // extern "C"
