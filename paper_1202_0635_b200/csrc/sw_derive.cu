// sw_derive_* of include/sw.h: the doubles the paper plots, from the integer histograms the kernels produce.
// Plain host code, no device work: the histograms are the measurement, these are fixed-order sums over at most 16 bins
// (d or k ascending, left to right, in double; R11, R15).  NaN on invalid arguments.
#include <cmath>
#include <cstdint>
#include <limits>

#include "sw.h"

namespace {

constexpr double kPi = 3.14159265358979323846;
const double kNaN = std::numeric_limits<double>::quiet_NaN();

inline bool q_ok(int q) { return q >= 2 && q <= SW_MAX_Q; }

// eq.(3): exact 64-bit integer numerator (N <= 2^28, q <= 16), one division
inline double m2_of(int q, const int64_t *n)
{
    int64_t total = 0, squares = 0;
    for (int k = 0; k < q; ++k) {
        total += n[k];
        squares += n[k] * n[k];
    }
    return (double)((int64_t)q * squares - total * total) / (double)(q - 1);
}

// eq.(5), one configuration: average of cos(2 pi d / q) over the counted pairs
inline double g_of(int q, const int64_t *c)
{
    double sum = 0.0;
    int64_t pairs = 0;
    for (int d = 0; d < q; ++d) {
        sum += (double)c[d] * std::cos(2.0 * kPi * (double)d / (double)q);
        pairs += c[d];
    }
    return sum / (double)pairs;
}

}  // namespace

extern "C" {

double sw_derive_potts_energy(int L, const int64_t *bond_hist)
{
    if (L < 2 || L > SW_MAX_L || !bond_hist) return kNaN;
    return (double)(2 * (int64_t)L * (int64_t)L - bond_hist[0]);
}

double sw_derive_potts_m2(int q, const int64_t *state_hist)
{
    if (!q_ok(q) || !state_hist) return kNaN;
    return m2_of(q, state_hist);
}

double sw_derive_clock_energy(int q, const int64_t *bond_hist)
{
    if (!q_ok(q) || !bond_hist) return kNaN;
    double e = 0.0;
    for (int d = 0; d < q; ++d) e += (double)bond_hist[d] * std::cos(2.0 * kPi * (double)d / (double)q);
    return -e;
}

double sw_derive_clock_m(int q, const int64_t *state_hist)
{
    if (!q_ok(q) || !state_hist) return kNaN;
    double mx = 0.0, my = 0.0;
    for (int k = 0; k < q; ++k) {
        mx += (double)state_hist[k] * std::cos(2.0 * kPi * (double)k / (double)q);
        my += (double)state_hist[k] * std::sin(2.0 * kPi * (double)k / (double)q);
    }
    return std::hypot(mx, my);
}

double sw_derive_g(int q, const int64_t *corr_hist)
{
    if (!q_ok(q) || !corr_hist) return kNaN;
    return g_of(q, corr_hist);
}

double sw_derive_moment_ratio(int n, int q, const int64_t *state_hist_rows)
{
    if (n < 1 || !q_ok(q) || !state_hist_rows) return kNaN;
    double sum2 = 0.0, sum4 = 0.0;
    for (int k = 0; k < n; ++k) {
        const double m2 = m2_of(q, state_hist_rows + (size_t)k * q);
        sum2 += m2;
        sum4 += m2 * m2;
    }
    const double mean2 = sum2 / (double)n;
    return (sum4 / (double)n) / (mean2 * mean2);
}

double sw_derive_ratio_R(int n, int q, const int64_t *corr_half_rows, const int64_t *corr_quarter_rows)
{
    if (n < 1 || !q_ok(q) || !corr_half_rows || !corr_quarter_rows) return kNaN;
    double half = 0.0, quarter = 0.0;
    for (int k = 0; k < n; ++k) {
        half += g_of(q, corr_half_rows + (size_t)k * q);
        quarter += g_of(q, corr_quarter_rows + (size_t)k * q);
    }
    return (half / (double)n) / (quarter / (double)n);
}

}  // extern "C"
