/*
 * oracle/ising_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU restatement of the hot path of
 * arxiv 2502.18624 (Bisson et al.): checkerboard Metropolis sweeps of the 2D
 * Ising (Eq. 1) and Blume-Capel (Eq. 2) models
 * on a periodic L x L lattice, integer observables and spin-spin correlation
 * sums (Sec. 3.3), Schwinger-Dyson sum (PAPER.md:182-189,
 * Eq. 3).  One int8 per spin, s[y*L + x], x = column, y = row.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code, header, table
 * or constant generator with paper_2502_18624_b200/csrc (the CUDA path).
 *
 * Every function follows the paper's algorithm step by step; where the paper
 * is silent the reading is the one listed in DESIGN.md "Readings" (R-numbers
 * below refer to that table).  Nothing here is blocked, fused or reordered.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer
 * vectors, closed-form thresholds, tally == recompute invariant, exact
 * enumeration of 4x4 Ising / 3x3 + 4x4 Blume-Capel, Onsager energy and
 * magnetisation, crafted-lattice closed forms for observables, brute force and
 * sum identities for correlation, Schwinger-Dyson -> 1; the row-band forms of
 * the observables and of the histogram (orc_observables_rows, orc_sd_hist_rows:
 * for lattices streamed out of the GPU in bands) by "the bands of any partition
 * add up to the full-lattice routine" and a python double loop; the time grid and
 * the Sec. 3.3 lists also by exact integer criteria (tests/test_oracle_correlation.py).  Section O7 (the
 * paper's 1-bit look-up-table kernel, tests/test_oracle_lut.py): table
 * marginals / independence / closed forms, getMaxLE against a library
 * search, per-word sweep == independently written per-site sweep, tally ==
 * recompute, 4x4 exact enumeration, Onsager.  No function is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_ISING 0
#define ORC_BC 1

/* ------------------------------------------------------------------ O1 --- */
/* Philox4x32-10 (the generator the paper names).  Ten rounds;
 * one round maps (c0,c1,c2,c3),(k0,k1) to
 *   (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0));
 * the key is bumped by the Weyl constants between rounds (9 bumps).        */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        if (round < 9) { k0 += W0; k1 += W1; }
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* draw(n, t, tag): the 32-bit uniform of colour-site index n (R3).
 * counter = (g_lo, g_hi, t, tag), key = (seed_lo, seed_hi), g = n >> 2,
 * output word n & 3.  tag: 0 black update, 1 white update, 2 black init,
 * 3 white init.                                                            */
uint32_t orc_draw(uint64_t seed, uint64_t n, uint32_t t, uint32_t tag)
{
    uint64_t g = n >> 2;
    uint32_t ctr[4] = { (uint32_t)(g & 0xFFFFFFFFu), (uint32_t)(g >> 32), t, tag };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    return out[n & 3];
}

/* colour-site index of lattice site (x, y): n = y*W + (x >> 1), W = (L+1)>>1 */
static inline uint64_t site_index(int64_t L, int64_t x, int64_t y)
{
    uint64_t W = (uint64_t)((L + 1) >> 1);
    return (uint64_t)y * W + (uint64_t)(x >> 1);
}

/* ------------------------------------------------------------------ O3 --- */
/* T = 2^32 if p >= 1 else floor(p * 2^32), p = exp(-beta*dE) in double (R4,R5).
 * A move is accepted iff (uint64)r < T, so P(accept) = T / 2^32 exactly.   */
static uint64_t threshold_of(double beta, double dE)
{
    double p = exp(-beta * dE);
    if (p >= 1.0) return 4294967296ull;
    return (uint64_t)floor(p * 4294967296.0);
}

/* Ising: index (dE+8)/4 for dE = 2*sigma*h in {-8,-4,0,4,8} (PAPER.md:93:
 * e^{-4 beta} with three equal neighbours, e^{-8 beta} with four, 1 else). */
static void ising_table(double beta, uint64_t T[5])
{
    for (int i = 0; i < 5; ++i) T[i] = threshold_of(beta, (double)(4 * i - 8));
}

/* Blume-Capel proposal (R8): uniform over the two other states, cyclic in the
 * code s+1: code' = (code + 1 + b) mod 3, b = r & 1.                       */
static inline int bc_proposal(int s, int b) { return ((s + 1) + 1 + b) % 3 - 1; }

/* Blume-Capel: index ((s+1)*2 + b)*9 + (h+4).  dE = D*dq - ds*h from Eq. 2
 * (J = 1): one multiply, one subtract.                                     */
static void bc_table(double beta, double D, uint64_t T[54])
{
    for (int s = -1; s <= 1; ++s)
        for (int b = 0; b <= 1; ++b)
            for (int h = -4; h <= 4; ++h) {
                int sp = bc_proposal(s, b);
                int ds = sp - s, dq = sp * sp - s * s;
                volatile double a = D * (double)dq;      /* no FMA contraction */
                double dE = a - (double)(ds * h);
                T[((s + 1) * 2 + b) * 9 + (h + 4)] = threshold_of(beta, dE);
            }
}

int orc_thresholds(int model, double beta, double D, uint64_t *out)
{
    if (model == ORC_ISING) { ising_table(beta, out); return 5; }
    bc_table(beta, D, out);
    return 54;
}

/* ------------------------------------------------------------------ O2 --- */
/* Init (R11).  Ising: sigma = +1 if top bit of r set else -1.  Blume-Capel:
 * code = (r*3) >> 32 in {0,1,2}, s = code - 1.  Patch form: fills the w x h
 * window whose top-left lattice site is (x0, y0), coordinates mod L.       */
void orc_init_patch(int model, int64_t L, uint64_t seed,
                    int64_t x0, int64_t y0, int64_t w, int64_t h, int8_t *s)
{
    for (int64_t j = 0; j < h; ++j)
        for (int64_t i = 0; i < w; ++i) {
            int64_t x = ((x0 + i) % L + L) % L, y = ((y0 + j) % L + L) % L;
            uint32_t c = (uint32_t)((x + y) & 1);
            uint32_t r = orc_draw(seed, site_index(L, x, y), 0u, 2u + c);
            if (model == ORC_ISING) s[j * w + i] = (r >> 31) ? 1 : -1;
            else s[j * w + i] = (int8_t)((int)(((uint64_t)r * 3u) >> 32) - 1);
        }
}

void orc_init(int model, int64_t L, uint64_t seed, int8_t *s)
{
    orc_init_patch(model, L, seed, 0, 0, L, L, s);
}

/* ------------------------------------------------------------------ O4 --- */
/* One Metropolis attempt at lattice site (x,y) whose four neighbours sum to h.
 * Updates *sp in place and the running tallies (bond sum B, M, Q).          */
static inline void attempt(int model, const uint64_t *T, uint32_t r, int h,
                           int8_t *sp, int64_t *B, int64_t *M, int64_t *Q)
{
    int s = *sp;
    if (model == ORC_ISING) {
        int dE = 2 * s * h;                     /* E = -B, flipping s changes B by -2*s*h */
        if ((uint64_t)r < T[(dE + 8) / 4]) {
            *B -= 2 * s * h; *M -= 2 * s; *sp = (int8_t)(-s);
        }
    } else {
        int b = (int)(r & 1u);
        int snew = bc_proposal(s, b);
        if ((uint64_t)r < T[((s + 1) * 2 + b) * 9 + (h + 4)]) {
            *B += (snew - s) * h; *Q += snew * snew - s * s; *M += snew - s;
            *sp = (int8_t)snew;
        }
    }
}

/* One full sweep number t (= sweeps completed before it, R "Sweep index"):
 * colour 0 = (x+y) even first, then colour 1 (R2).  Sites of a colour are
 * visited sequentially and updated in place.  tallies[3] = {B, M, Q} are
 * running values the caller initialised from orc_observables.
 * For even L no two same-colour sites are neighbours, so the rows of one
 * colour may be visited in any order (the OpenMP split below relies on that
 * and is disabled for odd L).                                              */
void orc_sweep(int model, int64_t L, double beta, double D, uint64_t seed,
               uint32_t t, int8_t *s, int64_t *tallies)
{
    uint64_t T[54];
    orc_thresholds(model, beta, D, T);
    int64_t B = tallies[0], M = tallies[1], Q = tallies[2];
    for (uint32_t c = 0; c < 2; ++c) {
        int64_t dB = 0, dM = 0, dQ = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : dB, dM, dQ) if ((L % 2) == 0 && L >= 64)
#endif
        for (int64_t y = 0; y < L; ++y) {
            int64_t ym = (y + L - 1) % L, yp = (y + 1) % L;
            for (int64_t x = (int64_t)((y + c) & 1); x < L; x += 2) {
                int64_t xm = (x + L - 1) % L, xp = (x + 1) % L;
                int h = s[ym * L + x] + s[yp * L + x] + s[y * L + xm] + s[y * L + xp];
                uint32_t r = orc_draw(seed, site_index(L, x, y), t, c);
                attempt(model, T, r, h, &s[y * L + x], &dB, &dM, &dQ);
            }
        }
        B += dB; M += dM; Q += dQ;
    }
    tallies[0] = B; tallies[1] = M; tallies[2] = Q;
}

/* Light-cone patch sweep: the same rule applied to the w x h window at (x0,y0)
 * (global coordinates mod L select the random numbers).  Neighbours outside
 * the window read as 0, so after n sweeps only sites at least 2n from the
 * window edge are exact (one site of contamination per half sweep).        */
void orc_sweep_patch(int model, int64_t L, double beta, double D, uint64_t seed,
                     uint32_t t, int64_t x0, int64_t y0, int64_t w, int64_t h, int8_t *s)
{
    uint64_t T[54];
    orc_thresholds(model, beta, D, T);
    /* rows of one colour are independent (no two same-colour sites are neighbours, L even): the row loop
     * may be split over threads exactly as in orc_sweep */
    for (uint32_t c = 0; c < 2; ++c) {
#ifdef _OPENMP
#pragma omp parallel for schedule(static) if ((L % 2) == 0 && h >= 16)
#endif
        for (int64_t j = 0; j < h; ++j)
            for (int64_t i = 0; i < w; ++i) {
                int64_t dump[3] = { 0, 0, 0 };
                int64_t x = ((x0 + i) % L + L) % L, y = ((y0 + j) % L + L) % L;
                if ((uint32_t)((x + y) & 1) != c) continue;
                int hs = 0;
                if (j > 0) hs += s[(j - 1) * w + i];
                if (j < h - 1) hs += s[(j + 1) * w + i];
                if (i > 0) hs += s[j * w + i - 1];
                if (i < w - 1) hs += s[j * w + i + 1];
                uint32_t r = orc_draw(seed, site_index(L, x, y), t, c);
                attempt(model, T, r, hs, &s[j * w + i], &dump[0], &dump[1], &dump[2]);
            }
    }
}

/* ------------------------------------------------------------------ O5 --- */
/* Full recompute (R12): every bond once, B = sum s(x,y)*(s(x+1,y)+s(x,y+1)),
 * M = sum s, Q = sum s^2.  out[3] = {B, M, Q}.                             */
void orc_observables(int64_t L, const int8_t *s, int64_t *out)
{
    int64_t B = 0, M = 0, Q = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : B, M, Q) if (L >= 1024)
#endif
    for (int64_t y = 0; y < L; ++y)
        for (int64_t x = 0; x < L; ++x) {
            int v = s[y * L + x];
            B += v * (s[y * L + (x + 1) % L] + s[((y + 1) % L) * L + x]);
            M += v; Q += v * v;
        }
    out[0] = B; out[1] = M; out[2] = Q;
}

/* The same sums restricted to the rows [y0, y0 + ny) of the lattice, for lattices the host cannot hold
 * (SURVEY.md Sec. 8(c) "Large-L parity": O5 applied to a lattice streamed out in row bands): band holds
 * ny + 1 rows of L spins -- the rows y0 .. y0 + ny, the last one (row (y0 + ny) mod L) only as the lower
 * neighbour of row y0 + ny - 1.  The bands of a partition of [0, L) add up to orc_observables.          */
void orc_observables_rows(int64_t L, int64_t ny, const int8_t *band, int64_t *out)
{
    int64_t B = 0, M = 0, Q = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : B, M, Q) if (L >= 1024)
#endif
    for (int64_t j = 0; j < ny; ++j)
        for (int64_t x = 0; x < L; ++x) {
            int v = band[j * L + x];
            B += v * (band[j * L + (x + 1) % L] + band[(j + 1) * L + x]);
            M += v; Q += v * v;
        }
    out[0] = B; out[1] = M; out[2] = Q;
}

/* Schwinger-Dyson histogram (Eq. 3) of the rows [y0, y0 + ny): band holds ny + 2 rows, the rows
 * y0 - 1 .. y0 + ny (mod L); hist[k+4] += #sites of the ny inner rows with s*h = k.                    */
void orc_sd_hist_rows(int64_t L, int64_t ny, const int8_t *band, int64_t *hist)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : hist[:9]) if (L >= 1024)
#endif
    for (int64_t j = 1; j <= ny; ++j)
        for (int64_t x = 0; x < L; ++x) {
            int h = band[(j - 1) * L + x] + band[(j + 1) * L + x]
                  + band[j * L + (x + L - 1) % L] + band[j * L + (x + 1) % L];
            hist[band[j * L + x] * h + 4] += 1;
        }
}

/* E = -B (Ising, Eq. 1) or -B + D*Q (Blume-Capel, Eq. 2; R10), J = 1.
 * out[4] = {E, E/N, M/N, (N-Q)/N}, one division each.                      */
void orc_normalised(int model, int64_t L, double D, const int64_t *bmq, double *out)
{
    double N = (double)L * (double)L;
    double E = (model == ORC_ISING) ? -(double)bmq[0] : -(double)bmq[0] + D * (double)bmq[2];
    out[0] = E; out[1] = E / N; out[2] = (double)bmq[1] / N;
    out[3] = ((double)(L * L - bmq[2])) / N;
}

/* Schwinger-Dyson (Eq. 3): hist[k+4] = #sites with sigma*h = k,
 * returns (1/N) sum_k hist[k+4] * exp(-2*beta*k).                          */
double orc_schwinger_dyson(int64_t L, double beta, const int8_t *s, int64_t *hist)
{
    for (int k = 0; k < 9; ++k) hist[k] = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : hist[:9]) if (L >= 1024)
#endif
    for (int64_t y = 0; y < L; ++y)
        for (int64_t x = 0; x < L; ++x) {
            int h = s[((y + L - 1) % L) * L + x] + s[((y + 1) % L) * L + x]
                  + s[y * L + (x + L - 1) % L] + s[y * L + (x + 1) % L];
            hist[s[y * L + x] * h + 4] += 1;
        }
    double acc = 0.0;
    for (int k = -4; k <= 4; ++k) acc += (double)hist[k + 4] * exp(-2.0 * beta * (double)k);
    return acc / ((double)L * (double)L);
}

/* ------------------------------------------------------------------ O6 --- */
/* Full-source pair sums (R13): S_x(r) = sum_{x,y} s(x,y) s(x+r,y),
 * S_y(r) = sum_{x,y} s(x,y) s(x,y+r), periodic, r = 1..rmax; entry r-1.     */
void orc_correlation(int64_t L, const int8_t *s, int64_t rmax, int64_t *sx, int64_t *sy)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int64_t r = 1; r <= rmax; ++r) {
        int64_t ax = 0, ay = 0;
        for (int64_t y = 0; y < L; ++y)
            for (int64_t x = 0; x < L; ++x) {
                int v = s[y * L + x];
                ax += v * s[y * L + (x + r) % L];
                ay += v * s[((y + r) % L) * L + x];
            }
        sx[r - 1] = ax; sy[r - 1] = ay;
    }
}

/* The same sums for an explicit list of distances and a source stride:
 * sources are the sites with x % stride == 0 and y % stride == 0 (R14).    */
void orc_correlation_list(int64_t L, const int8_t *s, int64_t stride,
                          int64_t count, const int64_t *r, int64_t *sx, int64_t *sy)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int64_t i = 0; i < count; ++i) {
        int64_t ax = 0, ay = 0, d = r[i];
        for (int64_t y = 0; y < L; y += stride)
            for (int64_t x = 0; x < L; x += stride) {
                int v = s[y * L + x];
                ax += v * s[y * L + (x + d) % L];
                ay += v * s[((y + d) % L) * L + x];
            }
        sx[i] = ax; sy[i] = ay;
    }
}

/* Sec. 3.3 protocol constants (R15, R16):
 * R = 16, r_c(t) = max{256, floor(g(L) sqrt(t) + 0.5)},
 * g(L) = 6 sqrt(ln(L / 2^16) / 3.3^2 + 1).                                  */
int64_t orc_protocol_rc(int64_t L, uint64_t t)
{
    double g = 6.0 * sqrt(log((double)L / 65536.0) / (3.3 * 3.3) + 1.0);
    int64_t rc = (int64_t)floor(g * sqrt((double)t) + 0.5);
    return rc < 256 ? 256 : rc;
}

/* Distance list at time t, in increasing order, clipped to L/2:
 *   r = 1..2R              (all sources,           stride[i] = 1)
 *   r = 2R+1..r_c(t)       (one source per RxR,    stride[i] = R)
 *   r in {floor(2^(x/32))} > r_c(t), x <= 32(log2 L - 1)   (stride[i] = R)
 * Returns the number of entries (writes at most cap of them).              */
int64_t orc_protocol_list(int64_t L, uint64_t t, int64_t cap, int64_t *r, int64_t *stride)
{
    const int64_t R = 16;
    int64_t half = L / 2, rc = orc_protocol_rc(L, t), n = 0;
    for (int64_t d = 1; d <= 2 * R && d <= half; ++d, ++n)
        if (n < cap) { r[n] = d; stride[n] = 1; }
    for (int64_t d = 2 * R + 1; d <= rc && d <= half; ++d, ++n)
        if (n < cap) { r[n] = d; stride[n] = R; }
    int64_t xmax = (int64_t)floor(32.0 * (log2((double)L) - 1.0) + 1e-9);
    int64_t last = (rc > 2 * R) ? rc : 2 * R;
    for (int64_t x = 0; x <= xmax; ++x) {
        int64_t d = (int64_t)floor(exp2((double)x / 32.0));
        if (d <= last || d > half) continue;
        if (n < cap) { r[n] = d; stride[n] = R; }
        ++n; last = d;
    }
    return n;
}

/* Measurement times t = floor(2^(x/8) + 0.5), x = 1,2,... (R17),
 * de-duplicated, t <= tmax.  Returns the count.                            */
int64_t orc_time_grid(uint64_t tmax, int64_t cap, uint64_t *out)
{
    int64_t n = 0; uint64_t last = 0;
    for (int x = 1; x < 8 * 64; ++x) {
        double v = floor(exp2((double)x / 8.0) + 0.5);
        if (v > (double)tmax) break;
        uint64_t t = (uint64_t)v;
        if (t == last) continue;
        if (n < cap) out[n] = t;
        ++n; last = t;
    }
    return n;
}

/* Thread count of the OpenMP loops (timing only: bench.py reports the oracle on all cores and on one). */
void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* n consecutive sweeps t0, t0+1, ...; trace (if non-NULL) receives {B, M, Q}
 * after each sweep (3*n int64).  Just the loop a caller would write.        */
void orc_run(int model, int64_t L, double beta, double D, uint64_t seed,
             uint32_t t0, int64_t n, int8_t *s, int64_t *tallies, int64_t *trace)
{
    for (int64_t i = 0; i < n; ++i) {
        orc_sweep(model, L, beta, D, seed, t0 + (uint32_t)i, s, tallies);
        if (trace) { trace[3 * i] = tallies[0]; trace[3 * i + 1] = tallies[1]; trace[3 * i + 2] = tallies[2]; }
    }
}

/* ================================================================== O7 === */
/* NEXT-2: the paper's own Ising kernel: one bit per spin, and
 * non-uniform random BITS from a look-up table instead of one uniform number
 * per spin.  Same acceptance probabilities as O4, a different trajectory
 * contract (readings L1-L6 in DESIGN.md):
 *
 *   flip = (eq4 & exp8) | (eq3 & exp4) | (~eq4 & ~eq3)
 *   exp4 = nonUniformRandBits();  exp8 = nonUniformRandBits() & exp4;
 *
 * where every bit of nonUniformRandBits() is 1 with probability p = e^{-4 beta},
 * so a spin with 4 equal neighbours flips with probability p^2 = e^{-8 beta}.
 * Four bits come from one 32-bit Philox number: getMaxLE(table, rnd) = the
 * largest index i in 0..15 with table[i] <= rnd, table[i] =
 * floor(2^32 * sum_{j<i} P(j)), P(j) = p^popc(j) (1-p)^(4-popc(j)).
 *
 * Keying (L3): the same-colour sites of a row are grouped in words of 64
 * (compact index k = x >> 1, word m = k >> 6, bit j = k & 63; Wr = ceil(L/128)
 * words per colour row, global word index w = y*Wr + m).  The 32 numbers of a
 * word come from 8 Philox calls with counter (g_lo, g_hi, t, colour), g = 8 w + q:
 * calls q = 0..3 feed exp4, q = 4..7 feed exp8; call q's output word u gives the
 * nibble 4 (q & 3) + u of its 64-bit word, i.e. bits 16 (q & 3) + 4 u + (0..3).   */

/* L2: the table in double, sums taken in index order; entries in [0, 2^32]. */
void orc_lut_table(double beta, uint64_t table[16])
{
    const double p = exp(-(4.0 * beta)), q = 1.0 - p;
    double pw[5], qw[5];
    pw[0] = 1.0; qw[0] = 1.0;
    for (int a = 1; a <= 4; ++a) { pw[a] = pw[a - 1] * p; qw[a] = qw[a - 1] * q; }
    double cum = 0.0;
    for (int i = 0; i < 16; ++i) {
        double v = floor(ldexp(cum, 32));
        if (v > 4294967296.0) v = 4294967296.0;
        table[i] = (uint64_t)v;
        const int ones = __builtin_popcount((unsigned)i);
        cum += pw[ones] * qw[4 - ones];
    }
}

static inline unsigned get_max_le(const uint64_t table[16], uint32_t rnd)
{
    unsigned idx = 0;
    for (unsigned i = 0; i < 16; ++i)
        if (table[i] <= (uint64_t)rnd) idx = i;      /* table is non-decreasing, table[0] = 0 */
    return idx;
}

static inline int64_t lut_words_per_row(int64_t L) { return (L / 2 + 63) / 64; }

/* The 64 random bits of word w: which = 0 -> exp4 source, 1 -> exp8 source.  */
uint64_t orc_lut_bits(const uint64_t table[16], uint64_t seed, uint64_t w, uint32_t t, uint32_t tag, int which)
{
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint64_t ret = 0;
    for (int k = 0; k < 64; k += 4) {                /* the paper's loop */
        const int nib = k / 4, q = which * 4 + nib / 4, u = nib % 4;
        const uint64_t g = 8 * w + (uint64_t)q;
        const uint32_t ctr[4] = { (uint32_t)g, (uint32_t)(g >> 32), t, tag };
        uint32_t out[4];
        orc_philox4x32_10(ctr, key, out);
        ret |= (uint64_t)get_max_le(table, out[u]) << k;
    }
    return ret;
}

/* L5: initial spins, one bit each: word w of colour c = (x | y << 32) of Philox(ctr = (w, t = 0, tag = 2 + c)). */
void orc_lut_init_patch(int64_t L, uint64_t seed, int64_t x0, int64_t y0, int64_t w, int64_t h, int8_t *s)
{
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    const int64_t Wr = lut_words_per_row(L);
    for (int64_t j = 0; j < h; ++j)
        for (int64_t i = 0; i < w; ++i) {
            const int64_t x = ((x0 + i) % L + L) % L, y = ((y0 + j) % L + L) % L;
            const uint32_t c = (uint32_t)((x + y) & 1);
            const int64_t k = x >> 1;
            const uint64_t wd = (uint64_t)(y * Wr + (k >> 6));
            const uint32_t ctr[4] = { (uint32_t)wd, (uint32_t)(wd >> 32), 0u, 2u + c };
            uint32_t out[4];
            orc_philox4x32_10(ctr, key, out);
            const uint64_t bits = (uint64_t)out[0] | ((uint64_t)out[1] << 32);
            s[j * w + i] = ((bits >> (k & 63)) & 1u) ? 1 : -1;
        }
}

void orc_lut_init(int64_t L, uint64_t seed, int8_t *s) { orc_lut_init_patch(L, seed, 0, 0, L, L, s); }

/* L4: one sweep in the paper's order: colour 0 then colour 1; for every word of 64 same-colour
 * sites the two random words are drawn, then each site applies the flip formula with its own
 * bit.  tallies = {B, M, Q} updated incrementally (E = -B).                                   */
void orc_lut_sweep(int64_t L, double beta, uint64_t seed, uint32_t t, int8_t *s, int64_t *tallies)
{
    uint64_t table[16];
    orc_lut_table(beta, table);
    const int64_t Wr = lut_words_per_row(L), half = L / 2;
    int64_t B = tallies[0], M = tallies[1];
    for (uint32_t c = 0; c < 2; ++c) {
        int64_t dB = 0, dM = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : dB, dM) if (L >= 64)
#endif
        for (int64_t y = 0; y < L; ++y) {
            const int64_t ym = (y + L - 1) % L, yp = (y + 1) % L, par = (y + c) & 1;
            for (int64_t m = 0; m < Wr; ++m) {
                const uint64_t w = (uint64_t)(y * Wr + m);
                const uint64_t exp4 = orc_lut_bits(table, seed, w, t, c, 0);
                const uint64_t exp8 = orc_lut_bits(table, seed, w, t, c, 1) & exp4;
                for (int j = 0; j < 64; ++j) {
                    const int64_t k = 64 * m + j;
                    if (k >= half) break;
                    const int64_t x = 2 * k + par, xm = (x + L - 1) % L, xp = (x + 1) % L;
                    const int sp = s[y * L + x];
                    const int h = s[ym * L + x] + s[yp * L + x] + s[y * L + xm] + s[y * L + xp];
                    const int eq = (4 + sp * h) / 2;             /* neighbours equal to the spin, 0..4 */
                    const int b4 = (int)((exp4 >> j) & 1u), b8 = (int)((exp8 >> j) & 1u);
                    const int flip = (eq == 4 && b8) || (eq == 3 && b4) || (eq <= 2);
                    if (flip) { dB -= 2 * sp * h; dM -= 2 * sp; s[y * L + x] = (int8_t)(-sp); }
                }
            }
        }
        B += dB; M += dM;
    }
    tallies[0] = B; tallies[1] = M;
}

/* Light-cone patch version, written per SITE (not per word): the bit of site (x, y) is looked
 * up from scratch, so it also serves as an independent restatement of the keying.            */
void orc_lut_sweep_patch(int64_t L, double beta, uint64_t seed, uint32_t t,
                         int64_t x0, int64_t y0, int64_t w, int64_t h, int8_t *s)
{
    uint64_t table[16];
    orc_lut_table(beta, table);
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    const int64_t Wr = lut_words_per_row(L);
    for (uint32_t c = 0; c < 2; ++c) {
#ifdef _OPENMP
#pragma omp parallel for schedule(static) if ((L % 2) == 0 && h >= 16)
#endif
        for (int64_t j = 0; j < h; ++j)
            for (int64_t i = 0; i < w; ++i) {
                const int64_t x = ((x0 + i) % L + L) % L, y = ((y0 + j) % L + L) % L;
                if ((uint32_t)((x + y) & 1) != c) continue;
                int hs = 0;
                if (j > 0) hs += s[(j - 1) * w + i];
                if (j < h - 1) hs += s[(j + 1) * w + i];
                if (i > 0) hs += s[j * w + i - 1];
                if (i < w - 1) hs += s[j * w + i + 1];
                const int64_t k = x >> 1, bit = k & 63;
                const uint64_t wd = (uint64_t)(y * Wr + (k >> 6));
                int b[2];
                for (int which = 0; which < 2; ++which) {
                    const uint64_t g = 8 * wd + (uint64_t)(which * 4 + bit / 16);
                    const uint32_t ctr[4] = { (uint32_t)g, (uint32_t)(g >> 32), t, c };
                    uint32_t out[4];
                    orc_philox4x32_10(ctr, key, out);
                    b[which] = (int)((get_max_le(table, out[(bit / 4) % 4]) >> (bit % 4)) & 1u);
                }
                const int sp = s[j * w + i];
                const int eq = (4 + sp * hs) / 2;
                const int flip = (eq == 4 && b[0] && b[1]) || (eq == 3 && b[0]) || (eq <= 2);
                if (flip) s[j * w + i] = (int8_t)(-sp);
            }
    }
}

/* n sweeps t0..t0+n-1 of the LUT kernel with the (B, M, Q) trace after each (test helper). */
void orc_lut_run(int64_t L, double beta, uint64_t seed, uint32_t t0, int64_t n, int8_t *s,
                 int64_t *tallies, int64_t *trace)
{
    for (int64_t i = 0; i < n; ++i) {
        orc_lut_sweep(L, beta, seed, t0 + (uint32_t)i, s, tallies);
        if (trace) { trace[3 * i] = tallies[0]; trace[3 * i + 1] = tallies[1]; trace[3 * i + 2] = tallies[2]; }
    }
}
