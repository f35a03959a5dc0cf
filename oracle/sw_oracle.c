/*
 * sw_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, sequential CPU statement of one Swendsen-Wang multi-cluster sweep of a 2D periodic
 * L x L lattice, written from arXiv 1202.0635 (Komura & Okabe), /root/reference/PAPER.md, in the
 * paper's order (PAPER.md:36-45 steps (i)-(viii)):  bonds -> cluster labels -> new state per
 * cluster -> spin update.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code, header, table or
 * helper with the CUDA path under paper_1202_0635_b200/csrc/.
 *
 * Where the paper is silent the readings of DESIGN.md section 3 (R1..R15) are used; each is
 * cited at its point of use.  Parity status: every function below is pinned by tests/ (Philox
 * known answers, high-precision thresholds, brute-force flood fill, exact enumeration of the
 * Boltzmann distribution on small tori, Kaufman/Onsager energy; oracle_correlation: tests/test_oracle_corr_pins.py;
 * the derived doubles oracle_potts_energy .. oracle_ratio_R: tests/test_oracle_derived_pins.py)
 * -- nothing is "parity unpinned".
 *
 * Conventions: N = L*L, site i = y*L + x (x fastest).  Each site owns two bonds:
 * direction 0 to (x+1 mod L, y) and direction 1 to (x, y+1 mod L)  (periodic; R8).
 * Spin states are 0..q-1 (paper: 1..q; R2).  J = 1.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_POTTS 0
#define ORACLE_CLOCK 1

/* ------------------------------------------------------------------------------------------- */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  R3: replaces the paper's LCG             */
/* (PAPER.md:69).  One round: two 32x32->64 products, a word permutation and a key XOR; the key  */
/* is bumped by the Weyl constants between rounds (not after the last).                         */
/* ------------------------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Random streams (R5: a pure function of (seed, sweep t, site, direction)).
 *   stream 0 BOND    counter (i>>1, t, 0, 0)  word 2*(i&1)+d   d = 0:+x, 1:+y
 *   stream 1 CLUSTER counter (r>>2, t, 1, 0)  word r&3         r = canonical root
 *   stream 2 AXIS    counter (0,    t, 2, 0)  word 0
 *   stream 3 INIT    counter (i>>2, 0, 3, 0)  word i&3
 * key = (seed low 32 bits, seed high 32 bits). */
static uint32_t stream_word(uint64_t seed, uint32_t c0, uint32_t t, uint32_t stream, int word)
{
    uint32_t ctr[4] = { c0, t, stream, 0u };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[word];
}

static uint32_t r_bond(uint64_t seed, uint32_t t, uint32_t i, int d)
{
    return stream_word(seed, i >> 1, t, 0u, (int)(2u * (i & 1u)) + d);
}
static uint32_t r_cluster(uint64_t seed, uint32_t t, uint32_t root)
{
    return stream_word(seed, root >> 2, t, 1u, (int)(root & 3u));
}
static uint32_t r_axis(uint64_t seed, uint32_t t)
{
    return stream_word(seed, 0u, t, 2u, 0);
}
static uint32_t r_init(uint64_t seed, uint32_t i)
{
    return stream_word(seed, i >> 2, 0u, 3u, (int)(i & 3u));
}

/* R6: a 32-bit word w becomes a state in [0,q) as floor(w*q / 2^32). */
static uint32_t mulhi_q(uint32_t w, uint32_t q)
{
    return (uint32_t)(((uint64_t)w * (uint64_t)q) >> 32);
}

/* Mirror axis of sweep t (clock model; R4: uniform over the q lattice-preserving reflections). */
uint32_t oracle_axis(int q, uint64_t seed, uint32_t t)
{
    return mulhi_q(r_axis(seed, t), (uint32_t)q);
}

/* ------------------------------------------------------------------------------------------- */
/* Thresholds (R6, R7): a bond is active iff r_bond < thr (unsigned, strict), thr =              */
/* floor(p * 2^32) clamped to 2^32 - 1, computed in double.                                      */
/* ------------------------------------------------------------------------------------------- */
static uint32_t thr_of_p(double p)
{
    double v = floor(p * 4294967296.0);
    if (!(v > 0.0)) return 0u;
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    return (uint32_t)v;
}

/* Potts, PAPER.md:37 step (ii) (garbled "p = 1 e^{-beta}"; R1: p = 1 - exp(-J/T), the reading
 * for which PAPER.md:75's Tc = 1/ln(1+sqrt q) is the self-dual point of eq.(1)). */
uint32_t oracle_potts_threshold(double T)
{
    return thr_of_p(1.0 - exp(-1.0 / T));
}

/* Clock, eq.(4) + Wolff's embedding (R4).  With mirror axis m the spin p has
 * c = (2p - m) mod 2q and component s(c) = sin(pi*c/q) along the mirror normal.  Reflecting one
 * end of a bond changes its energy by 2*J*s_i*s_j, so the embedded Ising bond is activated with
 * probability 1 - exp(-2*s_i*s_j/T) when s_i*s_j > 0, never otherwise.  s is exactly 0 on the
 * mirror line (c mod q == 0).  table has (2q)*(2q) entries, table[ci*2q + cj]. */
void oracle_clock_table(int q, double T, uint32_t *table)
{
    const double pi = 3.14159265358979323846;
    int n = 2 * q;
    for (int ci = 0; ci < n; ++ci) {
        for (int cj = 0; cj < n; ++cj) {
            double si = (ci % q == 0) ? 0.0 : sin(pi * (double)ci / (double)q);
            double sj = (cj % q == 0) ? 0.0 : sin(pi * (double)cj / (double)q);
            double prod = si * sj;
            table[ci * n + cj] = (prod > 0.0) ? thr_of_p(1.0 - exp(-2.0 * prod / T)) : 0u;
        }
    }
}

/* ------------------------------------------------------------------------------------------- */
/* Initial configuration (R12): S0_i = mulhi(word_INIT(i), q).                                   */
/* ------------------------------------------------------------------------------------------- */
void oracle_init_spins(int L, int q, uint64_t seed, uint8_t *spins)
{
    uint32_t N = (uint32_t)L * (uint32_t)L;
    for (uint32_t i = 0; i < N; ++i)
        spins[i] = (uint8_t)mulhi_q(r_init(seed, i), (uint32_t)q);
}

/* ------------------------------------------------------------------------------------------- */
/* Step 1 -- bond activation, PAPER.md:36-38 (i)-(iii).  bonds[i] bit0 = +x bond, bit1 = +y.     */
/* ------------------------------------------------------------------------------------------- */
int oracle_bonds(int L, int q, int model, double T, uint64_t seed, uint32_t t,
                 const uint8_t *spins, uint8_t *bonds)
{
    uint32_t N = (uint32_t)L * (uint32_t)L;
    uint32_t potts_thr = 0u, m = 0u;
    uint32_t *table = NULL;
    int n2 = 2 * q;
    if (model == ORACLE_POTTS) {
        potts_thr = oracle_potts_threshold(T);
    } else {
        table = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)n2 * (size_t)n2);
        if (!table) return -1;
        oracle_clock_table(q, T, table);
        m = oracle_axis(q, seed, t);
    }
    for (int y = 0; y < L; ++y) {
        for (int x = 0; x < L; ++x) {
            uint32_t i = (uint32_t)y * (uint32_t)L + (uint32_t)x;
            uint32_t nbr[2];
            nbr[0] = (uint32_t)y * (uint32_t)L + (uint32_t)((x + 1) % L);
            nbr[1] = (uint32_t)((y + 1) % L) * (uint32_t)L + (uint32_t)x;
            uint8_t b = 0;
            for (int d = 0; d < 2; ++d) {
                uint32_t thr;
                if (model == ORACLE_POTTS) {
                    thr = (spins[i] == spins[nbr[d]]) ? potts_thr : 0u;
                } else {
                    int ci = (int)((2u * spins[i] + (uint32_t)n2 - m) % (uint32_t)n2);
                    int cj = (int)((2u * spins[nbr[d]] + (uint32_t)n2 - m) % (uint32_t)n2);
                    thr = table[ci * n2 + cj];
                }
                if (r_bond(seed, t, i, d) < thr) b |= (uint8_t)(1u << d);
            }
            bonds[i] = b;
        }
    }
    (void)N;
    free(table);
    return 0;
}

/* ------------------------------------------------------------------------------------------- */
/* Step 2 -- cluster labeling, PAPER.md:39 (iv) and PAPER.md:47: "The proper label of a cluster  */
/* ... is defined to be the smallest label of any spin in the cluster ... found by evaluating     */
/* label[label] repeatedly."  Sequential union-find in the Hoshen-Kopelman spirit: parent         */
/* pointers always point to a smaller-or-equal index, so the fixed point of label[label] is the   */
/* minimum site index of the component.  On exit labels[i] = that minimum for every site.         */
/* ------------------------------------------------------------------------------------------- */
static int32_t proper_label(int32_t *label, int32_t a)
{
    while (label[a] != a) a = label[a];
    return a;
}

void oracle_label(int L, const uint8_t *bonds, int32_t *labels)
{
    int32_t N = (int32_t)L * (int32_t)L;
    for (int32_t i = 0; i < N; ++i) labels[i] = i;
    for (int y = 0; y < L; ++y) {
        for (int x = 0; x < L; ++x) {
            int32_t i = y * L + x;
            int32_t nbr[2];
            nbr[0] = y * L + (x + 1) % L;
            nbr[1] = ((y + 1) % L) * L + x;
            for (int d = 0; d < 2; ++d) {
                if (!((bonds[i] >> d) & 1)) continue;
                int32_t a = proper_label(labels, i);
                int32_t b = proper_label(labels, nbr[d]);
                if (a < b) labels[b] = a;
                else if (b < a) labels[a] = b;
            }
        }
    }
    /* i ascending: labels[labels[i]] is already final when site i is reached. */
    for (int32_t i = 0; i < N; ++i) labels[i] = proper_label(labels, i);
}

/* ------------------------------------------------------------------------------------------- */
/* Steps 3+4 -- new state per cluster and spin update, PAPER.md:40-42 (v)-(vii) and PAPER.md:69. */
/* Potts (R9): independent uniform redraw S'_i = mulhi(r_cluster(t, root), q).                    */
/* Clock (R4): cluster flipped iff top bit of r_cluster is set; flip = reflection                 */
/* p -> (m - p) mod q.                                                                            */
/* ------------------------------------------------------------------------------------------- */
void oracle_flip(int L, int q, int model, uint64_t seed, uint32_t t,
                 const int32_t *labels, uint8_t *spins)
{
    uint32_t N = (uint32_t)L * (uint32_t)L;
    uint32_t m = (model == ORACLE_CLOCK) ? oracle_axis(q, seed, t) : 0u;
    for (uint32_t i = 0; i < N; ++i) {
        uint32_t w = r_cluster(seed, t, (uint32_t)labels[i]);
        if (model == ORACLE_POTTS) {
            spins[i] = (uint8_t)mulhi_q(w, (uint32_t)q);
        } else if (w >> 31) {
            spins[i] = (uint8_t)((m + (uint32_t)q - spins[i]) % (uint32_t)q);
        }
    }
}

/* One full sweep t: S^t -> S^{t+1} (R10: axis -> bonds from S^t -> labels -> decisions).
 * labels_out / bonds_out may be NULL.  Returns 0, or -1 if memory could not be obtained. */
int oracle_sweep(int L, int q, int model, double T, uint64_t seed, uint32_t t,
                 uint8_t *spins, int32_t *labels_out, uint8_t *bonds_out)
{
    size_t N = (size_t)L * (size_t)L;
    uint8_t *bonds = bonds_out ? bonds_out : (uint8_t *)malloc(N);
    int32_t *labels = labels_out ? labels_out : (int32_t *)malloc(N * sizeof(int32_t));
    int rc = -1;
    if (bonds && labels && oracle_bonds(L, q, model, T, seed, t, spins, bonds) == 0) {
        oracle_label(L, bonds, labels);
        oracle_flip(L, q, model, seed, t, labels, spins);
        rc = 0;
    }
    if (!bonds_out) free(bonds);
    if (!labels_out) free(labels);
    return rc;
}

/* ------------------------------------------------------------------------------------------- */
/* Observables of a configuration ("+ measurement"; eq.(3); R11):        */
/* bond_hist[d] = number of owned bonds with (S_i - S_nbr) mod q == d; state_hist[k] = n[k].      */
/* ------------------------------------------------------------------------------------------- */
void oracle_observables(int L, int q, const uint8_t *spins, int64_t *bond_hist, int64_t *state_hist)
{
    for (int k = 0; k < q; ++k) { bond_hist[k] = 0; state_hist[k] = 0; }
    for (int y = 0; y < L; ++y) {
        for (int x = 0; x < L; ++x) {
            int s = spins[y * L + x];
            int sr = spins[y * L + (x + 1) % L];
            int sd = spins[((y + 1) % L) * L + x];
            bond_hist[((s - sr) % q + q) % q] += 1;
            bond_hist[((s - sd) % q + q) % q] += 1;
            state_hist[s] += 1;
        }
    }
}

/* Correlation histogram at distance r (eq.(5), eq.(6); R15):   */
/* corr_hist[d] = number of pairs (i, i + r e_x) and (i, i + r e_y), periodic, with (S_i - S_{i+r}) mod q  */
/* == d; 2N pairs.  G(r) = (1/2N) sum_d corr_hist[d] cos(2 pi d / q) is derived by the caller.             */
void oracle_correlation(int L, int q, const uint8_t *spins, int r, int64_t *corr_hist)
{
    for (int k = 0; k < q; ++k) corr_hist[k] = 0;
    for (int y = 0; y < L; ++y) {
        for (int x = 0; x < L; ++x) {
            int s = spins[y * L + x];
            int sx = spins[y * L + (x + r) % L];
            int sy = spins[((y + r) % L) * L + x];
            corr_hist[((s - sx) % q + q) % q] += 1;
            corr_hist[((s - sy) % q + q) % q] += 1;
        }
    }
}

/* ------------------------------------------------------------------------------------------- */
/* Derived doubles (R11, R15): what the paper plots, computed from the integer histograms in a    */
/* fixed order (sums run over d or k ascending, left to right, in double).                        */
/* ------------------------------------------------------------------------------------------- */
#define ORACLE_PI 3.14159265358979323846

/* Potts energy of eq.(1), in units of J: every owned bond with unequal spins costs 1. */
double oracle_potts_energy(int L, const int64_t *bond_hist)
{
    return (double)(2 * (int64_t)L * (int64_t)L - bond_hist[0]);
}

/* Eq.(3): M^2 = (q sum_k n[k]^2 - N^2) / (q - 1).  The numerator is an exact integer
 * (< 2^63 for N <= 2^28, q <= 16); one division in double. */
double oracle_potts_m2(int q, const int64_t *state_hist)
{
    int64_t N = 0, acc = 0;
    for (int k = 0; k < q; ++k) { N += state_hist[k]; acc += state_hist[k] * state_hist[k]; }
    return (double)((int64_t)q * acc - N * N) / (double)(q - 1);
}

/* Clock energy of eq.(4), in units of J: - sum over owned bonds of cos(theta_i - theta_j). */
double oracle_clock_energy(int q, const int64_t *bond_hist)
{
    double e = 0.0;
    for (int d = 0; d < q; ++d) e += (double)bond_hist[d] * cos(2.0 * ORACLE_PI * (double)d / (double)q);
    return -e;
}

/* |M| of the clock model: length of the vector sum of the planar unit spins. */
double oracle_clock_m(int q, const int64_t *state_hist)
{
    double mx = 0.0, my = 0.0;
    for (int k = 0; k < q; ++k) {
        mx += (double)state_hist[k] * cos(2.0 * ORACLE_PI * (double)k / (double)q);
        my += (double)state_hist[k] * sin(2.0 * ORACLE_PI * (double)k / (double)q);
    }
    return hypot(mx, my);
}

/* Eq.(5), for one configuration: G(r) = (1/pairs) sum over the counted pairs of S_i . S_{i+r}
 * = (1/pairs) sum_d corr_hist[d] cos(2 pi d / q)  (R15). */
double oracle_g(int q, const int64_t *corr_hist)
{
    double g = 0.0;
    int64_t pairs = 0;
    for (int d = 0; d < q; ++d) {
        g += (double)corr_hist[d] * cos(2.0 * ORACLE_PI * (double)d / (double)q);
        pairs += corr_hist[d];
    }
    return g / (double)pairs;
}

/* Eq.(2): U = <M^4> / <M^2>^2 over a recorded series of n state histograms (rows of q), M^2 of
 * every row by eq.(3), averages accumulated row by row. */
double oracle_moment_ratio(int n, int q, const int64_t *state_hist_rows)
{
    double s2 = 0.0, s4 = 0.0;
    for (int k = 0; k < n; ++k) {
        double m2 = oracle_potts_m2(q, state_hist_rows + (size_t)k * q);
        s2 += m2;
        s4 += m2 * m2;
    }
    return (s4 / (double)n) / ((s2 / (double)n) * (s2 / (double)n));
}

/* Eq.(6): R = <G(L/2)> / <G(L/4)>, the averages of eq.(5) over a recorded series of n
 * correlation histograms at the two distances (rows of q). */
double oracle_ratio_R(int n, int q, const int64_t *corr_half_rows, const int64_t *corr_quarter_rows)
{
    double gh = 0.0, gq = 0.0;
    for (int k = 0; k < n; ++k) {
        gh += oracle_g(q, corr_half_rows + (size_t)k * q);
        gq += oracle_g(q, corr_quarter_rows + (size_t)k * q);
    }
    return (gh / (double)n) / (gq / (double)n);
}

/* n sweeps t0 .. t0+n-1.  If bond_rec/state_rec are non-NULL, row k (q entries each) receives
 * the observables of the configuration BEFORE sweep t0+k (R10). */
int oracle_run(int L, int q, int model, double T, uint64_t seed, uint32_t t0, int n,
               uint8_t *spins, int64_t *bond_rec, int64_t *state_rec)
{
    for (int k = 0; k < n; ++k) {
        if (bond_rec && state_rec)
            oracle_observables(L, q, spins, bond_rec + (size_t)k * q, state_rec + (size_t)k * q);
        if (oracle_sweep(L, q, model, T, seed, t0 + (uint32_t)k, spins, NULL, NULL) != 0) return -1;
    }
    return 0;
}
