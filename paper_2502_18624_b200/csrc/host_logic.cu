// Host-only arithmetic of the path (no CUDA call in this file, so every entry point here runs
// and is tested on a machine without a GPU):
//   A1   acceptance thresholds floor(min(1, e^{-beta dE}) 2^32)
//   L2   the 16-entry cumulative table of the 1-bit kernel's getMaxLE
//   A11  the measurement times t = floor(2^{x/8} + 1/2)
//   A10  the Sec. 3.3 distance lists: all sources up to 2R, one source per R x R block up to
//        r_c(t), then the logarithmic grid floor(2^{x/32}) up to L/2
// Written from the paper's formulas; tests/test_host_logic.py pins each of them to values the
// mathematics fixes (exact integer criteria, 60-digit decimals, tests/golden/protocol_pins.txt).
#include <math.h>

#include <algorithm>
#include <vector>

#include "ising_internal.cuh"

// ------------------------------------------------------------ thresholds ---
// A1: T = 2^32 if p >= 1 else floor(p 2^32), p = exp(-beta dE) evaluated in double.
static uint64_t metropolis_threshold(double beta, double dE)
{
    const double p = exp(-(beta * dE));
    if (p >= 1.0) return 1ull << 32;
    return (uint64_t)floor(ldexp(p, 32));
}

// Reading L2: pattern j of four independent bits, each 1 with probability p = e^{-4 beta}, has
// probability P(j) = p^k (1 - p)^(4 - k), k = popcount(j); entry i of the table is floor(2^32 C_i) with
// C_i = P(0) + ... + P(i - 1) accumulated in index order in double (powers by repeated multiplication,
// every product and sum rounded once -- the rounding order is part of the reading, both sides follow it).
static void lut_cumulative_table(double beta, uint64_t T[16])
{
    const double p1 = exp(-(4.0 * beta)), p0 = 1.0 - p1;
    double ones[5], zeros[5];                      // p1^k, p0^k
    ones[0] = zeros[0] = 1.0;
    for (int k = 1; k <= 4; ++k) { ones[k] = ones[k - 1] * p1; zeros[k] = zeros[k - 1] * p0; }
    double per_class[5];                           // probability of ONE pattern with k bits set
    for (int k = 0; k <= 4; ++k) {
        volatile double prod = ones[k] * zeros[4 - k];     // rounded product (no FMA into the sum below)
        per_class[k] = prod;
    }
    double below = 0.0;                            // C_i
    for (unsigned i = 0; i < 16; ++i) {
        // 2^32 C_i is exact in double (a power-of-two scaling); C_i can exceed 1 by a rounding error only
        T[i] = below >= 1.0 ? (1ull << 32) : (uint64_t)(below * 4294967296.0);
        below += per_class[__builtin_popcount(i)];
    }
}

int host_threshold_table(int model, double beta, double D, uint64_t *T)
{
    if (model == ISING_MODEL_ISING_LUT) { lut_cumulative_table(beta, T); return 16; }
    if (model == ISING_MODEL_ISING) {
        // entry i: dE = 2 s h = 4 i - 8 in {-8,-4,0,4,8}
        for (int i = 0; i < 5; ++i) T[i] = metropolis_threshold(beta, 4.0 * i - 8.0);
        return 5;
    }
    // Blume-Capel (Eq. 2): single-site energy e(s) = -s h + D s^2
    for (int code = 0; code < 3; ++code)
        for (int b = 0; b < 2; ++b)
            for (int S = 0; S <= 8; ++S) {
                const int s_old = code - 1, s_new = (code + 1 + b) % 3 - 1, field = S - 4;
                const int d_lin = (s_new - s_old) * field;                 // change of s h
                const int d_sq = s_new * s_new - s_old * s_old;            // change of s^2
                volatile double crystal = D * (double)d_sq;                // rounded product, no FMA
                const double dE = crystal - (double)d_lin;
                T[(code * 2 + b) * 9 + S] = metropolis_threshold(beta, dE);
            }
    return 54;
}

static bool known_model(int model)
{
    return model == ISING_MODEL_ISING || model == ISING_MODEL_BLUME_CAPEL || model == ISING_MODEL_ISING_LUT ||
           model == ISING_MODEL_BLUME_CAPEL_2BIT;
}

extern "C" int ising_threshold_table(int model, double beta, double D, uint64_t *out, int cap, int *count)
{
    if (!count) return set_error(ISING_EINVAL, "ising_threshold_table: count is NULL");
    if (!known_model(model)) return set_error(ISING_EINVAL, "ising_threshold_table: unknown model");
    if (!(beta >= 0.0) || !isfinite(beta) || !isfinite(D)) return set_error(ISING_EINVAL, "ising_threshold_table: beta must be finite and >= 0, D finite");
    uint64_t T[54];
    const int n = host_threshold_table(model, beta, is_blume_capel(model) ? D : 0.0, T);
    *count = n;
    if (!out) return ISING_OK;                                  // size query
    if (cap < n) return set_error(ISING_EINVAL, "ising_threshold_table: cap too small");
    for (int i = 0; i < n; ++i) out[i] = T[i];
    return ISING_OK;
}

// ---------------------------------------------------- powers 2^(x / 2^k) ---
// 2^(x / 2^K) = 2^q * prod_{bits b of j} 2^(2^b / 2^K), x = q 2^K + j: the K fractional factors are K nested
// square roots of 2 (correctly rounded), so the value is exact when j = 0 and within a few ulp otherwise.
template <int K>
struct DyadicPowers {
    double root[K];                                // root[b] = 2^(2^b / 2^K)
    DyadicPowers()
    {
        double v = 2.0;
        for (int b = K - 1; b >= 0; --b) { v = sqrt(v); root[b] = v; }
    }
    double operator()(int64_t x) const
    {
        const int64_t q = x >> K, j = x & ((1 << K) - 1);
        double f = 1.0;
        for (int b = 0; b < K; ++b)
            if ((j >> b) & 1) f *= root[b];
        return ldexp(f, (int)q);
    }
};

// ---------------------------------------------------------------- A11 ------
// Measurement times of the paper: t_x = 2^(x/8) rounded to the nearest integer, x = 1, 2, ...;
// neighbouring x give the same t while 2^(x/8) < 12, so equal times are listed once.
void host_time_grid(uint64_t tmax, std::vector<uint64_t> &times)
{
    static const DyadicPowers<3> eighth_powers;
    times.clear();
    for (int64_t x = 1; x < 8 * 63; ++x) {
        const double nearest = floor(eighth_powers(x) + 0.5);
        if (nearest > (double)tmax) break;
        const uint64_t t = (uint64_t)nearest;
        if (times.empty() || times.back() != t) times.push_back(t);
    }
}

extern "C" int ising_time_grid(uint64_t tmax, uint64_t *out, int64_t cap, int64_t *count)
{
    if (!count) return set_error(ISING_EINVAL, "ising_time_grid: count is NULL");
    std::vector<uint64_t> times;
    host_time_grid(tmax, times);
    *count = (int64_t)times.size();
    if (!out) return ISING_OK;                                  // size query
    if (cap < *count) return set_error(ISING_EINVAL, "ising_time_grid: cap too small");
    std::copy(times.begin(), times.end(), out);
    return ISING_OK;
}

// ---------------------------------------------------------------- A10 ------
// Sec. 3.3.  R = 16.  Distances 1..2R use every site as a source; beyond that one source
// per R x R block: every r up to the crossover r_c(t) = max{256, [g(L) sqrt(t)]} ([.] = nearest integer),
// g(L) = 6 sqrt(ln(L / 2^16) / 3.3^2 + 1) (natural logarithm, reading R16), then the logarithmic grid
// floor(2^(x/32)), x = 0, 1, 2, ..., as long as 2^(x/32) <= L/2 (reading R15: "32 values of r for each power
// of two, up to L/2"), keeping the values above r_c, each once.  Everything is clipped to L/2.
static const int64_t kBlock = 16;                  // R

int64_t host_protocol_crossover(int64_t L, uint64_t t)
{
    const double ratio = (double)L / 65536.0;
    const double g = 6.0 * sqrt(log(ratio) / (3.3 * 3.3) + 1.0);
    const int64_t nearest = (int64_t)floor(g * sqrt((double)t) + 0.5);
    return std::max<int64_t>(256, nearest);
}

void host_protocol_lists(int64_t L, uint64_t t, std::vector<int64_t> &all_sources, std::vector<int64_t> &block_sources)
{
    static const DyadicPowers<5> thirty_second_powers;
    const int64_t reach = L / 2, rc = host_protocol_crossover(L, t);
    all_sources.clear();
    block_sources.clear();
    for (int64_t r = 1; r <= std::min(2 * kBlock, reach); ++r) all_sources.push_back(r);
    for (int64_t r = 2 * kBlock + 1; r <= std::min(rc, reach); ++r) block_sources.push_back(r);
    int64_t largest = std::max(rc, 2 * kBlock);    // the grid continues above what is already listed
    for (int64_t x = 0;; ++x) {
        const double v = thirty_second_powers(x);
        if (v > (double)reach) break;
        const int64_t r = (int64_t)floor(v);
        if (r > largest) { block_sources.push_back(r); largest = r; }
    }
}

extern "C" int ising_protocol_distances(int64_t L, uint64_t t, int64_t cap, int64_t *r, int64_t *stride, int64_t *count)
{
    if (!count) return set_error(ISING_EINVAL, "ising_protocol_distances: count is NULL");
    if (L < 2 || (L & 1) || L > (1ll << 40)) return set_error(ISING_EINVAL, "ising_protocol_distances: L must be even, in [2, 2^40]");
    std::vector<int64_t> all_sources, block_sources;
    host_protocol_lists(L, t, all_sources, block_sources);
    const int64_t na = (int64_t)all_sources.size(), nb = (int64_t)block_sources.size();
    *count = na + nb;
    if (!r && !stride) return ISING_OK;                         // size query
    if (!r || !stride || cap < na + nb) return set_error(ISING_EINVAL, "ising_protocol_distances: cap too small");
    for (int64_t i = 0; i < na; ++i) { r[i] = all_sources[i]; stride[i] = 1; }
    for (int64_t i = 0; i < nb; ++i) { r[na + i] = block_sources[i]; stride[na + i] = kBlock; }
    return ISING_OK;
}

// ---------------------------------------------------------------- NEXT-4 ---
// Default row partition of ising_create_slabs ("horizontal slabs"): the L/2 row pairs dealt as
// evenly as possible, so every slab starts on an even row and has an even height (a row pair is the unit the
// kernels walk: the row parity alternates inside it).
extern "C" int ising_slab_partition(int64_t L, int n_slabs, int64_t *rows)
{
    if (!rows) return set_error(ISING_EINVAL, "ising_slab_partition: rows is NULL");
    if (L < 2 || (L & 1) || n_slabs < 1 || n_slabs > ISING_MAX_SLABS || 2 * (int64_t)n_slabs > L)
        return set_error(ISING_EINVAL, "ising_slab_partition: L must be even and n_slabs in [1, min(64, L/2)]");
    const int64_t pairs = L / 2;
    for (int k = 0; k < n_slabs; ++k) rows[k] = 2 * (pairs * (k + 1) / n_slabs - pairs * k / n_slabs);
    return ISING_OK;
}
