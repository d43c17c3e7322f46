// hough_oracle_next.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain CPU restatement of the rows SURVEY.md 8(f) marks NEXT, written beside (not into) the pinned S1..S6 of
// hough_oracle.cpp, which stays untouched:
//   N1  candidate-circle / track-parameter epilogue      PAPER.md:77 Eq. (2), :150-158 (pT, phi0)
//   N2  paper-form peak finding: threshold relative to the global accumulator maximum + iterative
//       "extract the most significant peak, suppress its neighbourhood"
//   N4a theta wrap-around with the mirrored rho index ((theta + pi, rho) == (theta, -rho))
//   N4b original-space distance filter | ||hit - centre|| - r_c | < tol
// (N3, the paper's 1000 x 1000 grid, needs no new arithmetic: it is oracle_run with that grid.)
// Where the paper is silent the readings Q14..Q20 of DESIGN.md are taken; each function says which.
// Same build as hough_oracle.cpp (-ffp-contract=off: every operation rounds once, as written), linked into the same
// liboracle.so.  Shares no code with paper_2607_04067_b200/.  S1 and S2 are restated here (conformal, rho_bin) so
// that the pinned file needs no edit; tests/test_oracle_next_pins.py checks the two copies against each other.
//
// Pins (tests/test_oracle_next_pins.py): the closed-form circle P1 (r_c = 1644.31 mm, centre direction theta_40, the
// mirrored circle, the charge of either turning sense, phi0 within one theta bin of the generated one), the hand-worked
// rows of tests/golden/w1_next.txt (circle of peak (2,4), NMS order, wrapped neighbours), exact rescaling (scale 2),
// brute-force restatements in numpy, and invariants (NMS peaks are >= 1 + radius apart, descending votes, a subset of
// the cells >= threshold; wrap off == plain S3/S5; tol -> infinity keeps every hit of an event with a peak).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

struct ParamsX {
    int n_theta, n_rho;
    float rho_max, inv;
    int threshold, window, max_peaks;
    float scale;
    int acc_u16;
    const float* cos_t;
    const float* sin_t;
    // NEXT options
    int peak_mode;        // 0: threshold + 3x3 local maximum (S3); 1: relative threshold + iterative NMS (N2)
    int rel_permille;     // N2: cells below ceil(rel_permille * A_max / 1000) are no candidates (reading Q18)
    int nms_radius;       // N2: half-width of the suppressed neighbourhood, in bins
    int theta_wrap;       // N4a: column -1 is column n_theta-1 with the rho index mirrored (reading Q19)
    int keep_mode;        // 0: (theta, rho) window (S5); 1: distance to the candidate circle (N4b, reading Q20)
    double keep_tol;      // N4b: tolerance, units of the hit coordinates
    double b_field;       // N1: tesla
};

// S1 restated (Eq. (1)).
inline void conformal(float x, float y, float scale, float* u, float* v) {
    float xx = x * x;
    float yy = y * y;
    float d = xx + yy;
    float u1 = x / d;
    float v1 = y / d;
    *u = scale * u1;
    *v = scale * v1;
}

// S2 restated (readings Q4, Q5).  Returns k or -1.
inline int rho_bin(float u, float v, float c, float s, const ParamsX& p) {
    float uc = u * c;
    float vs = v * s;
    float rho = uc + vs;
    float shifted = rho + p.rho_max;
    float t = shifted * p.inv;
    if (t >= 0.0f && t < (float)p.n_rho) return (int)t;
    return -1;
}

void accumulate(const float* xy, int n_hits, const ParamsX& p, uint32_t* A) {
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

// N4a (reading Q19).  rho(theta + pi) = -rho(theta), so the column "before" theta_0 is the last column
// read upside down: (j, k) with j = -1 is (n_theta-1, n_rho-1-k), and j = n_theta is (0, n_rho-1-k).  Without wrap a
// cell outside the array is 0 (reading Q8).  Only one step beyond either border is ever mapped per n_theta columns,
// so |j| offsets up to n_theta are folded column by column.
inline bool fold(const ParamsX& p, int& j, int& k) {
    if (k < 0 || k >= p.n_rho) return false;
    if (j >= 0 && j < p.n_theta) return true;
    if (!p.theta_wrap) return false;
    while (j < 0) { j += p.n_theta; k = p.n_rho - 1 - k; }
    while (j >= p.n_theta) { j -= p.n_theta; k = p.n_rho - 1 - k; }
    return true;
}

inline uint32_t cell(const uint32_t* A, const ParamsX& p, int j, int k) {
    if (!fold(p, j, k)) return 0u;
    return A[(size_t)j * p.n_rho + k];
}

// S3 + S4 with the optional wrap: identical to hough_oracle.cpp's find_peaks when theta_wrap == 0.
int find_peaks_3x3(const uint32_t* A, const ParamsX& p, uint32_t* peaks_out) {
    int n_peaks = 0;
    for (int j = 0; j < p.n_theta; ++j) {
        for (int k = 0; k < p.n_rho; ++k) {
            uint32_t a = A[(size_t)j * p.n_rho + k];
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

// N2 (reading Q18).  "A relative threshold can be set according to the global maximum value of the
// accumulation matrix ... After extracting the current significant peak, it suppresses its local neighborhood and
// continues to search for the remaining independent peaks."
//   thr_eff = max(threshold, ceil(rel_permille * A_max / 1000))            (integers; threshold stays the floor)
//   repeat: take the largest remaining cell, the raster-first one among equals; stop if it is < thr_eff (or 0);
//           record it; set every cell within +-nms_radius bins in theta and rho (clipped, or folded when
//           theta_wrap is on) to 0.
// Peaks come out in extraction order (descending votes); the first max_peaks are stored, all are counted.
// W is a working copy of the accumulator (destroyed).
int find_peaks_nms(uint32_t* W, const ParamsX& p, uint32_t* peaks_out) {
    const size_t cells = (size_t)p.n_theta * p.n_rho;
    uint32_t a_max = 0;
    for (size_t c = 0; c < cells; ++c) if (W[c] > a_max) a_max = W[c];
    unsigned long long rel = ((unsigned long long)p.rel_permille * a_max + 999ull) / 1000ull;
    unsigned long long thr_eff = (unsigned long long)p.threshold > rel ? (unsigned long long)p.threshold : rel;
    int n_peaks = 0;
    for (;;) {
        uint32_t best = 0;
        size_t best_c = 0;
        for (size_t c = 0; c < cells; ++c) if (W[c] > best) { best = W[c]; best_c = c; }   // strict >: raster-first among equals
        if (best == 0 || (unsigned long long)best < thr_eff) break;
        int j = (int)(best_c / p.n_rho), k = (int)(best_c % p.n_rho);
        if (n_peaks < p.max_peaks) {
            peaks_out[3 * n_peaks + 0] = (uint32_t)j;
            peaks_out[3 * n_peaks + 1] = (uint32_t)k;
            peaks_out[3 * n_peaks + 2] = best;
        }
        ++n_peaks;
        for (int dj = -p.nms_radius; dj <= p.nms_radius; ++dj)
            for (int dk = -p.nms_radius; dk <= p.nms_radius; ++dk) {
                int jj = j + dj, kk = k + dk;
                if (fold(p, jj, kk)) W[(size_t)jj * p.n_rho + kk] = 0u;
            }
    }
    return n_peaks;
}

// S5 with the optional wrap (reading Q19): the window column j_p + dj beyond a border is the folded column, where the
// hit's own bin is compared with the MIRRORED peak bin.  Identical to hough_oracle.cpp's select_hits without wrap.
void select_hits_window(const float* xy, int n_hits, const ParamsX& p, const uint32_t* peaks, int n_stored, uint8_t* keep) {
    for (int i = 0; i < n_hits; ++i) {
        float u, v;
        conformal(xy[2 * i], xy[2 * i + 1], p.scale, &u, &v);
        uint8_t kp = 0;
        for (int q = 0; q < n_stored && !kp; ++q) {
            int jp = (int)peaks[3 * q + 0];
            int kpk = (int)peaks[3 * q + 1];
            for (int dj = -p.window; dj <= p.window; ++dj) {
                int j = jp + dj, kref = kpk;
                if (!fold(p, j, kref)) continue;        // kref becomes n_rho-1-k_p once per fold
                int k = rho_bin(u, v, p.cos_t[j], p.sin_t[j], p);
                if (k < 0) continue;
                int dk = k - kref; if (dk < 0) dk = -dk;
                if (dk <= p.window) { kp = 1; break; }
            }
        }
        keep[i] = kp;
    }
}

// N1 (Eq. (2); readings Q14-Q16).  The line rho = u cos(theta) + v sin(theta) of the conformal plane is
// the circle through the origin with centre (cos theta, sin theta) * s / (2 rho) and radius s / (2 |rho|), s the
// conformal scale: s = 2 is Eq. (2) as printed (x_c = cos/rho, r_c = 1/|rho|), s = 1 goes with Eq. (1) as printed
// (reading Q1).  rho is taken at the CENTRE of the peak's bin, all in fp64, one rounding per operation:
//   rho_c = (k + 0.5) / inv - rho_max
//   x_c = (s * c_j) / (2 * rho_c),  y_c = (s * s_j) / (2 * rho_c),  r_c = s / (2 * |rho_c|)   (IEEE: rho_c = 0 -> inf / NaN)
//   pT = (0.0003 * B) * r_c      [GeV/c for coordinates in mm and B in tesla: pT = 0.3 B R, R in m; PAPER.md:150]
struct Circle { double x_c, y_c, r_c, pt, phi0; int32_t charge, n_hits; };

inline double rho_centre(int k, const ParamsX& p) {
    double kc = (double)k + 0.5;
    double q = kc / (double)p.inv;
    return q - (double)p.rho_max;
}

inline void circle_of(int j, int k, const ParamsX& p, double* x_c, double* y_c, double* r_c) {
    double rc = rho_centre(k, p);
    double den = 2.0 * rc;
    double s = (double)p.scale;
    double nx = s * (double)p.cos_t[j];
    double ny = s * (double)p.sin_t[j];
    *x_c = nx / den;
    *y_c = ny / den;
    *r_c = s / std::fabs(den);
}

// N1, second half (reading Q17).  The circle alone does not say which way the particle turns; the
// hits do.  A hit is ASSOCIATED with the peak iff its own bin at the peak's column j_p is valid and within the keep
// window of k_p.  For an associated hit the fp32 cross product  z = c_j * y - s_j * x  (centre direction x hit) times
// the sign of rho_c says on which side of the centre direction it lies; n_pos / n_neg count the two sides.
//   charge = +1 if n_neg > n_pos, -1 if n_pos > n_neg, 0 on a tie     (+1: hits clockwise of the centre direction)
//   phi_c  = theta_j (+ pi if rho_c < 0),  theta_j = j * pi / n_theta           (azimuth of the centre, reading Q3)
//   phi0   = phi_c - charge * pi/2, folded into [0, 2 pi)     (direction of motion at the origin; the centre is at
//            phi0 + charge * pi/2, the convention of the input recipe)
void circles(const float* xy, int n_hits, const ParamsX& p, const uint32_t* peaks, int n_stored, Circle* out) {
    const double pi = 3.14159265358979323846;
    for (int q = 0; q < n_stored; ++q) {
        int j = (int)peaks[3 * q + 0], k = (int)peaks[3 * q + 1];
        Circle c;
        circle_of(j, k, p, &c.x_c, &c.y_c, &c.r_c);
        double kfac = 0.0003 * p.b_field;
        c.pt = kfac * c.r_c;
        double rc = rho_centre(k, p);
        int n_pos = 0, n_neg = 0, n_assoc = 0;
        for (int i = 0; i < n_hits; ++i) {
            float x = xy[2 * i], y = xy[2 * i + 1], u, v;
            conformal(x, y, p.scale, &u, &v);
            int kb = rho_bin(u, v, p.cos_t[j], p.sin_t[j], p);
            if (kb < 0) continue;
            int dk = kb - k; if (dk < 0) dk = -dk;
            if (dk > p.window) continue;
            ++n_assoc;
            float a = p.cos_t[j] * y;
            float b = p.sin_t[j] * x;
            float z = a - b;
            if (rc < 0.0) z = -z;
            if (z > 0.0f) ++n_pos;
            else if (z < 0.0f) ++n_neg;
        }
        c.n_hits = n_assoc;
        c.charge = n_neg > n_pos ? 1 : (n_pos > n_neg ? -1 : 0);
        double jt = (double)j * pi;
        double phi_c = jt / (double)p.n_theta;
        if (rc < 0.0) phi_c = phi_c + pi;
        double phi0 = phi_c - (double)c.charge * (pi / 2.0);
        if (phi0 < 0.0) phi0 = phi0 + 2.0 * pi;
        if (phi0 >= 2.0 * pi) phi0 = phi0 - 2.0 * pi;
        c.phi0 = phi0;
        out[q] = c;
    }
}

// N4b ("inversely mapped back to the original space through Eq. (2), and data filtering can then be
// performed on this basis"; :44 "candidate-circle parameters are geometrically associated with detector hits";
// reading Q20).  keep_i = 1 iff some STORED peak's circle has | sqrt((x-x_c)^2 + (y-y_c)^2) - r_c | < tol, fp64, one
// rounding per operation, sqrt correctly rounded.  A peak with rho_c = 0 (infinite radius) keeps nothing (NaN < tol is false).
void select_hits_distance(const float* xy, int n_hits, const ParamsX& p, const uint32_t* peaks, int n_stored, uint8_t* keep) {
    for (int i = 0; i < n_hits; ++i) {
        double x = (double)xy[2 * i], y = (double)xy[2 * i + 1];
        uint8_t kp = 0;
        for (int q = 0; q < n_stored && !kp; ++q) {
            double x_c, y_c, r_c;
            circle_of((int)peaks[3 * q + 0], (int)peaks[3 * q + 1], p, &x_c, &y_c, &r_c);
            double dx = x - x_c, dy = y - y_c;
            double dx2 = dx * dx, dy2 = dy * dy;
            double d = std::sqrt(dx2 + dy2);
            double e = std::fabs(d - r_c);
            if (e < p.keep_tol) kp = 1;
        }
        keep[i] = kp;
    }
}

void run_event_ex(const float* xy_all, int off, int n_hits, const ParamsX& p, uint8_t* keep_all, uint32_t* peaks_ev,
                  int32_t* counts_ev, float* kept_xy_all, int32_t* kept_idx_all, uint32_t* accum_out, Circle* circles_ev,
                  std::vector<uint32_t>& scratch, std::vector<uint32_t>& work) {
    if (p.acc_u16 && n_hits > 65535) { counts_ev[0] = -1; counts_ev[1] = -1; return; }
    const float* xy = xy_all + 2 * (size_t)off;
    uint32_t* A = accum_out;
    if (!A) { scratch.resize((size_t)p.n_theta * p.n_rho); A = scratch.data(); }
    accumulate(xy, n_hits, p, A);
    int n_peaks;
    if (p.peak_mode == 1) {
        work.assign(A, A + (size_t)p.n_theta * p.n_rho);     // the dump keeps the votes; suppression works on a copy
        n_peaks = find_peaks_nms(work.data(), p, peaks_ev);
    } else {
        n_peaks = find_peaks_3x3(A, p, peaks_ev);
    }
    int n_stored = n_peaks < p.max_peaks ? n_peaks : p.max_peaks;
    uint8_t* keep = keep_all + off;
    if (p.keep_mode == 1) select_hits_distance(xy, n_hits, p, peaks_ev, n_stored, keep);
    else select_hits_window(xy, n_hits, p, peaks_ev, n_stored, keep);
    int m = 0;
    for (int i = 0; i < n_hits; ++i) {
        if (keep[i]) {
            if (kept_xy_all) { kept_xy_all[2 * (size_t)(off + m)] = xy[2 * i]; kept_xy_all[2 * (size_t)(off + m) + 1] = xy[2 * i + 1]; }
            if (kept_idx_all) kept_idx_all[off + m] = i;
            ++m;
        }
    }
    counts_ev[0] = n_peaks;
    counts_ev[1] = m;
    if (circles_ev) circles(xy, n_hits, p, peaks_ev, n_stored, circles_ev);
}

}  // namespace

extern "C" {

// oracle_run with the NEXT options.  opts = {peak_mode, rel_permille, nms_radius, theta_wrap, keep_mode}; circles
// [n_events][max_peaks] x 48 bytes {x_c, y_c, r_c, pt, phi0 (fp64), charge, n_hits (int32)} may be null.
int oracle_run_ex(const float* xy, const int32_t* offsets, int n_events, int n_theta, int n_rho, float rho_max, int threshold,
                  int window, int max_peaks, int conformal_scale, int acc_u16, const float* cos_t, const float* sin_t,
                  const int32_t* opts, double keep_tol, double b_field, uint8_t* keep, uint32_t* peaks, int32_t* counts,
                  float* kept_xy, int32_t* kept_idx, uint32_t* accum, void* circles_out, int n_threads) {
    if (n_theta < 1 || n_rho < 1 || !(rho_max > 0.0f) || threshold < 1 || window < 0 || max_peaks < 0 || n_events < 0) return -1;
    if (conformal_scale != 1 && conformal_scale != 2) return -1;
    if (opts[0] < 0 || opts[0] > 1 || opts[1] < 0 || opts[1] > 1000 || opts[2] < 0 || opts[4] < 0 || opts[4] > 1) return -1;
    ParamsX p;
    p.n_theta = n_theta; p.n_rho = n_rho; p.rho_max = rho_max;
    p.inv = (float)((double)n_rho / (2.0 * (double)rho_max));
    p.threshold = threshold; p.window = window; p.max_peaks = max_peaks;
    p.scale = (float)conformal_scale; p.acc_u16 = acc_u16; p.cos_t = cos_t; p.sin_t = sin_t;
    p.peak_mode = opts[0]; p.rel_permille = opts[1]; p.nms_radius = opts[2]; p.theta_wrap = opts[3]; p.keep_mode = opts[4];
    p.keep_tol = keep_tol; p.b_field = b_field;
    Circle* circ = (Circle*)circles_out;
    auto range = [&](int e0, int e1) {
        std::vector<uint32_t> scratch, work;
        for (int e = e0; e < e1; ++e) {
            int off = offsets[e];
            run_event_ex(xy, off, offsets[e + 1] - off, p, keep, peaks + (size_t)e * max_peaks * 3, counts + 2 * (size_t)e, kept_xy,
                         kept_idx, accum ? accum + (size_t)e * n_theta * n_rho : nullptr,
                         circ ? circ + (size_t)e * max_peaks : nullptr, scratch, work);
        }
    };
    if (n_threads <= 1 || n_events <= 1) {
        range(0, n_events);
    } else {
        if (n_threads > n_events) n_threads = n_events;
        std::vector<std::thread> pool;
        for (int t = 0; t < n_threads; ++t)
            pool.emplace_back(range, (int)((long long)n_events * t / n_threads), (int)((long long)n_events * (t + 1) / n_threads));
        for (auto& th : pool) th.join();
    }
    return 0;
}

// Peak finding alone, on a caller-made accumulator A [n_theta][n_rho] (so that a pin can hand-craft plateaus, borders
// and seams).  opts as in oracle_run_ex; returns n_peaks (untruncated), peaks_out [max_peaks][3].
int oracle_find_peaks_ex(const uint32_t* A, int n_theta, int n_rho, int threshold, int max_peaks, const int32_t* opts, uint32_t* peaks_out) {
    ParamsX p{};
    p.n_theta = n_theta; p.n_rho = n_rho; p.threshold = threshold; p.max_peaks = max_peaks;
    p.peak_mode = opts[0]; p.rel_permille = opts[1]; p.nms_radius = opts[2]; p.theta_wrap = opts[3];
    if (p.peak_mode == 1) {
        std::vector<uint32_t> w(A, A + (size_t)n_theta * n_rho);
        return find_peaks_nms(w.data(), p, peaks_out);
    }
    return find_peaks_3x3(A, p, peaks_out);
}

}  // extern "C"
