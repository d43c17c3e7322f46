// gen.cpp -- seeded synthetic STCF-MDC-shaped events (inputs only).
//
// This module serves both the CPU oracle and the CUDA path with the SAME
// arrays; it holds none of the method's arithmetic (no conformal map, no Hough
// bins).  The recipe is stated in DESIGN.md "Input recipe" and follows
// BASELINE.json `configs` / SURVEY.md section 8(d):
//   * 2-D drift chamber, 48 layers at r_l = 200 + l*600/47 mm, B = 1 T,
//     R[mm] = 1000 * pT[GeV] / (0.3 * B);
//   * signal tracks are circles through the origin: pT log-uniform, phi0
//     uniform in [0, 2pi), charge q = +-1, centre direction phi_c = phi0 + q*pi/2,
//     one hit per layer with r_l <= 2R at azimuth phi_c - q*acos(r_l / 2R)
//     (outgoing branch), independent N(0, sigma = 0.13 mm) smears on x and y;
//     a track's hit set may be repeated `turns` times with fresh smears;
//   * background: Poisson(lambda) hits, uniform layer, uniform phi, exactly on
//     the layer radius;
//   * the hits of an event are Fisher-Yates shuffled;
//   * all maths in double, rounded once to fp32.
// Random numbers: SplitMix64, one stream per event seeded from (seed, event
// index), so that events are reproducible independently and in any chunking.
// Draw order per event: n_tracks; per track pT, phi0, q, turns, then per turn
// and layer dx, dy; n_bkg; per background hit layer, phi; shuffle.
#include <cmath>
#include <cstdint>
#include <utility>
#include <vector>

namespace {

struct SplitMix64 {
    uint64_t s;
    uint64_t next() {
        uint64_t z = (s += 0x9E3779B97F4A7C15ull);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        return z ^ (z >> 31);
    }
    double uniform() { return (double)(next() >> 11) * (1.0 / 9007199254740992.0); }          // [0,1)
    double uniform_open() { return ((double)(next() >> 11) + 1.0) * (1.0 / 9007199254740992.0); }  // (0,1]
    int below(int n) { int r = (int)(uniform() * (double)n); return r < n ? r : n - 1; }     // {0..n-1}
    double normal() {   // Box-Muller, cosine branch only: two uniforms per draw
        double u1 = uniform_open();
        double u2 = uniform();
        return std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586476925 * u2);
    }
    int poisson_knuth(double lambda) {   // lambda <= 32
        double L = std::exp(-lambda), p = 1.0;
        int k = 0;
        do { ++k; p *= uniform(); } while (p > L);
        return k - 1;
    }
    int poisson(double lambda) {         // sum of Poisson(<= 32) chunks
        int n = 0;
        while (lambda > 32.0) { n += poisson_knuth(32.0); lambda -= 32.0; }
        if (lambda > 0.0) n += poisson_knuth(lambda);
        return n;
    }
};

const int N_LAYERS = 48;
inline double layer_radius(int l) { return 200.0 + (double)l * 600.0 / 47.0; }

struct Hit { float x, y; uint8_t truth; };

}  // namespace

extern "C" {

// Generates events [first_event, first_event + n_events).  xy_out [cap][2]
// fp32 (mm), truth_out [cap] u8 (0 = background, t+1 = t-th track of the
// event), offsets_out [n_events+1] int32 (CSR, starts at 0).  Returns the
// total number of hits; if it exceeds `cap`, nothing beyond cap is written and
// the caller retries with a larger buffer (offsets_out is complete either way).
long long stcf_generate(unsigned long long seed, long long first_event, int n_events,
                        int tracks_lo, int tracks_hi, double pt_lo_gev, double pt_hi_gev,
                        int turns_lo, int turns_hi, double bkg_lambda, double sigma_mm,
                        float* xy_out, unsigned char* truth_out, long long cap, int* offsets_out) {
    const double PI = 3.14159265358979323846;
    long long total = 0;
    std::vector<Hit> ev;
    offsets_out[0] = 0;
    for (int e = 0; e < n_events; ++e) {
        uint64_t idx = (uint64_t)(first_event + e);
        SplitMix64 boot{seed * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull};
        uint64_t a = boot.next();
        SplitMix64 rng{a ^ (idx * 0xD1B54A32D192ED03ull + 0x2545F4914F6CDD1Dull)};
        rng.next();
        ev.clear();
        int n_tracks = tracks_lo + rng.below(tracks_hi - tracks_lo + 1);
        for (int t = 0; t < n_tracks; ++t) {
            double pt = pt_lo_gev * std::exp(rng.uniform() * std::log(pt_hi_gev / pt_lo_gev));
            double phi0 = 2.0 * PI * rng.uniform();
            double q = rng.below(2) ? 1.0 : -1.0;
            int turns = turns_lo + rng.below(turns_hi - turns_lo + 1);
            double R = 1000.0 * pt / 0.3;
            double phic = phi0 + q * PI / 2.0;
            for (int turn = 0; turn < turns; ++turn) {
                for (int l = 0; l < N_LAYERS; ++l) {
                    double r = layer_radius(l);
                    if (r > 2.0 * R) continue;
                    double phi = phic - q * std::acos(r / (2.0 * R));
                    double dx = sigma_mm * rng.normal();
                    double dy = sigma_mm * rng.normal();
                    Hit h;
                    h.x = (float)(r * std::cos(phi) + dx);
                    h.y = (float)(r * std::sin(phi) + dy);
                    h.truth = (uint8_t)(t + 1);
                    ev.push_back(h);
                }
            }
        }
        int n_bkg = rng.poisson(bkg_lambda);
        for (int b = 0; b < n_bkg; ++b) {
            int l = rng.below(N_LAYERS);
            double phi = 2.0 * PI * rng.uniform();
            double r = layer_radius(l);
            Hit h;
            h.x = (float)(r * std::cos(phi));
            h.y = (float)(r * std::sin(phi));
            h.truth = 0;
            ev.push_back(h);
        }
        for (int i = (int)ev.size() - 1; i > 0; --i) {   // Fisher-Yates
            int j = rng.below(i + 1);
            std::swap(ev[i], ev[j]);
        }
        for (size_t i = 0; i < ev.size(); ++i) {
            long long pos = total + (long long)i;
            if (pos < cap) {
                xy_out[2 * pos + 0] = ev[i].x;
                xy_out[2 * pos + 1] = ev[i].y;
                truth_out[pos] = ev[i].truth;
            }
        }
        total += (long long)ev.size();
        offsets_out[e + 1] = (int)total;
    }
    return total;
}

}  // extern "C"
