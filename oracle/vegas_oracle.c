/*
 * vegas_oracle.c -- plain, slow, single-threaded CPU Vegas.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the parity oracle of the repository.  It is NOT part of the product:
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call it.  It shares no code, header, table or constant
 * generator with paper_2002_12921_b200/csrc (the CUDA path) and neither includes the other.
 *
 * What it follows.  /root/reference/PAPER.md says only that the algorithm "is importance
 * sampling as implemented in Vegas [1, 2]" (section 2.2) with a per-event step
 * and an after-iteration step that "refine[s] how the random numbers are generated"
 * (PAPER.md:49-51), and gives the toy integrands (Eqs. (1)-(3)).  Every
 * numerical convention the paper leaves open is fixed by BASELINE.json:north_star and by the
 * readings C1..C9 of SURVEY.md section 8(c), restated in DESIGN.md ("Readings of the paper").
 * Each function below names the reading it implements, in the paper's order:
 *   per event: RNG (C1,C2) -> split (C3) -> grid map + Jacobian (C4) -> integrand (C5)
 *              -> accumulate S1, S2, H (C6);
 *   per iteration: estimate (C7), refine (C8);  per run: combine (C9).
 * No blocking, fusion, vectorisation or reordering: one event at a time, one dimension at a
 * time.  Floating point is fp64 (the fp32 GPU variant is compared against THIS fp64 oracle,
 * north_star: "the fp32 path must agree with the fp64 oracle to <=1e-5 relative");
 * the sums S1, S2 and H are carried in long double (x87 80-bit) so that summation order
 * cannot matter at the 1e-10 level (C6).
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): Philox known-answer vectors (C1), layout
 * vectors (C2), exact-rational split/map checks (C3, C4), closed forms by erf / atan and
 * independent quadrature of f (C5), brute-force re-accumulation in numpy and the Sum_b H = S2
 * invariant (C6, C7), fixed points / interp-based rebin / worked examples (C8), closed forms
 * (C9), 5-sigma agreement of whole chains with the closed-form integrals.
 *
 * Variants (readings C3' and C4' of DESIGN.md section 2), selected by the `variant` bit mask of
 * the *_v functions (0 = the method as above; the functions without _v are variant 0):
 *   ORACLE_V_U53 (1)  C3': 53-bit uniforms, two Philox words per draw (oracle_word53, oracle_split53);
 *   ORACLE_V_Q32 (2)  C4': the per-bin pair (X_b, Delta_b) of the sampling map rounded to fp32 (oracle_q32); the
 *                     master grid and the refinement stay fp64.
 * Pins: tests/test_oracle_variants.py (exact rationals for the 53-bit split and for the rounded map, an independent
 * Python-integer Philox for the two-word layout, brute-force re-accumulation, 5-sigma chains).
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared (see oracle/build.py).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ENUMERIC (-3)

#define ORACLE_MAX_DIM 64

#define ORACLE_V_U53 1
#define ORACLE_V_Q32 2

enum { F_CONST = 0, F_GAUSS = 1, F_GENZ_PRODUCT_PEAK = 2, F_BW_POLY = 3, F_GENZ_DISCONTINUOUS = 4 };

/* ---------------------------------------------------------------------------------------
 * C1  Philox4x32-10 (north_star: "counter-based Philox4x32-10 stream").
 * One round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * M0 = 0xD2511F53, M1 = 0xCD9E8D57; the key is bumped by (0x9E3779B9, 0xBB67AE85)
 * between rounds (9 bumps for 10 rounds).
 * ------------------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(prod1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)prod1;
        uint32_t n2 = (uint32_t)(prod0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)prod0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* C2  the 32-bit word of (seed, iteration, event e, dimension j):
 * key = (seed lo, seed hi); counter = (j>>2, iteration, e lo, e hi); word = output[j&3]. */
uint32_t oracle_word(uint64_t seed, uint32_t iteration, uint64_t event, int j)
{
    uint32_t ctr[4] = { (uint32_t)(j >> 2), iteration, (uint32_t)(event & 0xFFFFFFFFu),
                        (uint32_t)(event >> 32) };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[j & 3];
}

/* C3  split: P = word*nb exactly (64 bit); bin b = P>>32; lo = P & 0xFFFFFFFF;
 * r = (lo + 0.5) * 2^-32, exact in fp64, r in (0,1). */
void oracle_split(uint32_t word, int n_bins, int32_t *bin, double *r)
{
    uint64_t P = (uint64_t)word * (uint64_t)(uint32_t)n_bins;
    uint32_t lo = (uint32_t)(P & 0xFFFFFFFFu);
    *bin = (int32_t)(P >> 32);
    *r = ((double)lo + 0.5) * (1.0 / 4294967296.0);
}

/* C3' (variant ORACLE_V_U53)  53-bit uniforms from two words per draw.  One Philox block serves TWO dimensions:
 * key = (seed lo, seed hi); counter = (j>>1, iteration, e lo, e hi); dimension j takes hi = output[2(j&1)],
 * lo = output[2(j&1)+1] and U = hi * 2^21 + (lo >> 11), a 53-bit integer (the usual construction of a double in
 * [0,1) from two 32-bit words). */
uint64_t oracle_word53(uint64_t seed, uint32_t iteration, uint64_t event, int j)
{
    uint32_t ctr[4] = { (uint32_t)(j >> 1), iteration, (uint32_t)(event & 0xFFFFFFFFu),
                        (uint32_t)(event >> 32) };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    uint64_t hi = out[2 * (j & 1)], lo = out[2 * (j & 1) + 1];
    return (hi << 21) | (lo >> 11);
}

/* C3' split: P = U*nb exactly (U < 2^53, nb <= 256: P < 2^61); bin b = P >> 53; frac = P mod 2^53;
 * r = frac * 2^-53, exact in fp64, r in [0,1). */
void oracle_split53(uint64_t U, int n_bins, int32_t *bin, double *r)
{
    uint64_t P = U * (uint64_t)(uint32_t)n_bins;
    uint64_t frac = P & ((1ull << 53) - 1ull);
    *bin = (int32_t)(P >> 53);
    *r = (double)frac * (1.0 / 9007199254740992.0);
}

/* C4' (variant ORACLE_V_Q32)  a grid-table entry rounded to fp32 (round to nearest even) and widened back. */
double oracle_q32(double v)
{
    volatile float q = (float)v;
    return (double)q;
}

/* C5  built-in integrands, fp64 formulas.
 *   id 1  PAPER.md:65 Eq.(1), N = (a sqrt(pi))^-d    params = { a }
 *   id 2  PAPER.md:74 Eq.(3), N = 1                  params = { c[0..d-1], w[0..d-1] }
 *   id 3  BASELINE.json:configs[4] (reading R11,R12) params = { M, Gamma, m_min, m_max,
 *                                                               a[i][k], i=1..d-1, k=0..4 }
 *   id 4  PAPER.md:69 Eq.(2) AS PRINTED, N = 1 (reading R19): f = 0 if any x_j <= a_j, otherwise
 *         exp(sum_j c_j x_j)                         params = { c[0..d-1], a[0..d-1] }
 *   id 0  f = 1 */
int oracle_n_params(int integrand_id, int dim)
{
    switch (integrand_id) {
    case F_CONST: return 0;
    case F_GAUSS: return 1;
    case F_GENZ_PRODUCT_PEAK: return 2 * dim;
    case F_BW_POLY: return 4 + 5 * (dim - 1);
    case F_GENZ_DISCONTINUOUS: return 2 * dim;
    default: return -1;
    }
}

double oracle_f(int integrand_id, int dim, const double *x, const double *params)
{
    switch (integrand_id) {
    case F_CONST:
        return 1.0;
    case F_GAUSS: {
        const double pi = 3.14159265358979323846;
        double a = params[0];
        double norm = pow(a * sqrt(pi), -(double)dim);
        double sum = 0.0;
        for (int j = 0; j < dim; ++j) {
            double t = x[j] - 0.5;
            sum += t * t;
        }
        return norm * exp(-sum / (a * a));
    }
    case F_GENZ_PRODUCT_PEAK: {
        const double *c = params, *w = params + dim;
        double prod = 1.0;
        for (int j = 0; j < dim; ++j) {
            double t = x[j] - w[j];
            prod *= 1.0 / (c[j] * c[j]) + t * t;
        }
        return 1.0 / prod;
    }
    case F_BW_POLY: {
        double M = params[0], G = params[1], m_min = params[2], m_max = params[3];
        const double *a = params + 4;               /* a[(i-1)*5 + k], i = 1..dim-1 */
        double s_min = m_min * m_min, s_max = m_max * m_max;
        double s = s_min + x[0] * (s_max - s_min);
        double M2 = M * M, MG2 = M2 * G * G;
        double bw = MG2 / ((s - M2) * (s - M2) + MG2);
        double poly = 0.0;
        for (int i = 1; i < dim; ++i) {
            double xi = x[i], pw = 1.0;
            for (int k = 0; k < 5; ++k) {
                poly += a[(i - 1) * 5 + k] * pw;
                pw *= xi;
            }
        }
        return bw * poly;
    }
    case F_GENZ_DISCONTINUOUS: {
        const double *c = params, *a = params + dim;
        double sum = 0.0;
        for (int j = 0; j < dim; ++j) {
            if (x[j] <= a[j]) return 0.0;
            sum += c[j] * x[j];
        }
        return exp(sum);
    }
    default:
        return NAN;
    }
}

static int check_grid(int dim, int n_bins, const double *edges)
{
    if (dim < 1 || dim > ORACLE_MAX_DIM || n_bins < 2 || !edges) return ORACLE_EINVAL;
    for (int j = 0; j < dim; ++j) {
        const double *X = edges + (size_t)j * (n_bins + 1);
        for (int i = 0; i < n_bins; ++i)
            if (!(X[i + 1] > X[i])) return ORACLE_EINVAL;
    }
    return ORACLE_OK;
}

/* C2..C5 for ONE event: words, bins, x (C4: x_j = X[j][b] + (X[j][b+1]-X[j][b]) * r),
 * Jacobian J = prod_j n_bins * Delta_j, and f(x).  edges is [dim][n_bins+1], row-major. */
int oracle_sample_event_v(int variant, int dim, int n_bins, const double *edges, uint64_t seed,
                          uint32_t iteration, uint64_t event, int integrand_id,
                          const double *params, uint32_t *words, int32_t *bins, double *x,
                          double *jac, double *f)
{
    double J = 1.0;
    for (int j = 0; j < dim; ++j) {
        const double *X = edges + (size_t)j * (n_bins + 1);
        int32_t b;
        double r;
        if (variant & ORACLE_V_U53) {               /* C3': words[j] reports the top 32 bits of U */
            uint64_t U = oracle_word53(seed, iteration, event, j);
            oracle_split53(U, n_bins, &b, &r);
            if (words) words[j] = (uint32_t)(U >> 21);
        } else {
            uint32_t word = oracle_word(seed, iteration, event, j);
            oracle_split(word, n_bins, &b, &r);
            if (words) words[j] = word;
        }
        double x0 = X[b], delta = X[b + 1] - X[b];
        if (variant & ORACLE_V_Q32) {               /* C4': the table entry (X_b, Delta_b) in fp32 */
            x0 = oracle_q32(x0);
            delta = oracle_q32(delta);
        }
        x[j] = x0 + delta * r;
        J *= (double)n_bins * delta;
        bins[j] = b;
    }
    *jac = J;
    *f = oracle_f(integrand_id, dim, x, params);
    return ORACLE_OK;
}

int oracle_sample_event(int dim, int n_bins, const double *edges, uint64_t seed,
                        uint32_t iteration, uint64_t event, int integrand_id,
                        const double *params, uint32_t *words, int32_t *bins, double *x,
                        double *jac, double *f)
{
    return oracle_sample_event_v(0, dim, n_bins, edges, seed, iteration, event, integrand_id, params,
                                 words, bins, x, jac, f);
}

/* debug view of a range of events (parity hook for the CUDA K4 kernel, P1/P2):
 * words [count][dim], bins [count][dim], x [count][dim], fJ [count]. */
int oracle_sample_v(int variant, int dim, int n_bins, const double *edges, uint64_t seed, uint32_t iteration,
                    uint64_t first_event, uint64_t count, int integrand_id, const double *params,
                    uint32_t *words, int32_t *bins, double *x, double *fJ)
{
    int rc = check_grid(dim, n_bins, edges);
    if (rc) return rc;
    if (oracle_n_params(integrand_id, dim) < 0 || (variant & ~3)) return ORACLE_EINVAL;
    for (uint64_t q = 0; q < count; ++q) {
        double J, f;
        oracle_sample_event_v(variant, dim, n_bins, edges, seed, iteration, first_event + q, integrand_id,
                              params, words ? words + q * dim : NULL, bins + q * dim,
                              x + q * dim, &J, &f);
        fJ[q] = f * J;
    }
    return ORACLE_OK;
}

int oracle_sample(int dim, int n_bins, const double *edges, uint64_t seed, uint32_t iteration,
                  uint64_t first_event, uint64_t count, int integrand_id, const double *params,
                  uint32_t *words, int32_t *bins, double *x, double *fJ)
{
    return oracle_sample_v(0, dim, n_bins, edges, seed, iteration, first_event, count, integrand_id, params,
                           words, bins, x, fJ);
}

/* C6  accumulate events [first_event, first_event+count): v = f*J; S1 += v; S2 += v*v;
 * H[j][b_j] += v*v for every j.  Accumulators are long double; they are returned as
 * (hi, lo) double pairs (hi = (double)S, lo = (double)(S - hi)) so that disjoint event
 * ranges run by independent callers can be added without losing the extra bits.
 * sums = { S1_hi, S1_lo, S2_hi, S2_lo }; hist_hi / hist_lo are [dim][n_bins]. */
int oracle_accumulate_v(int variant, int dim, int n_bins, const double *edges, uint64_t seed,
                        uint32_t iteration, uint64_t first_event, uint64_t count,
                        int integrand_id, const double *params, double *sums, double *hist_hi,
                        double *hist_lo)
{
    int rc = check_grid(dim, n_bins, edges);
    if (rc) return rc;
    if (oracle_n_params(integrand_id, dim) < 0 || (variant & ~3)) return ORACLE_EINVAL;
    size_t nh = (size_t)dim * n_bins;
    long double *H = (long double *)calloc(nh, sizeof(long double));
    if (!H) return ORACLE_EINVAL;
    long double S1 = 0.0L, S2 = 0.0L;
    int32_t bins[ORACLE_MAX_DIM];
    double x[ORACLE_MAX_DIM];
    for (uint64_t q = 0; q < count; ++q) {
        double J, f;
        oracle_sample_event_v(variant, dim, n_bins, edges, seed, iteration, first_event + q, integrand_id,
                              params, NULL, bins, x, &J, &f);
        double v = f * J;
        double v2 = v * v;
        S1 += (long double)v;
        S2 += (long double)v2;
        for (int j = 0; j < dim; ++j) H[(size_t)j * n_bins + bins[j]] += (long double)v2;
    }
    sums[0] = (double)S1; sums[1] = (double)(S1 - (long double)sums[0]);
    sums[2] = (double)S2; sums[3] = (double)(S2 - (long double)sums[2]);
    for (size_t i = 0; i < nh; ++i) {
        hist_hi[i] = (double)H[i];
        if (hist_lo) hist_lo[i] = (double)(H[i] - (long double)hist_hi[i]);
    }
    free(H);
    return ORACLE_OK;
}

int oracle_accumulate(int dim, int n_bins, const double *edges, uint64_t seed,
                      uint32_t iteration, uint64_t first_event, uint64_t count,
                      int integrand_id, const double *params, double *sums, double *hist_hi,
                      double *hist_lo)
{
    return oracle_accumulate_v(0, dim, n_bins, edges, seed, iteration, first_event, count, integrand_id,
                               params, sums, hist_hi, hist_lo);
}

/* C7  estimate from the sums of n events: I = S1/n; Var = (S2/n - I^2)/(n-1);
 * sigma = sqrt(max(Var,0)).  Inputs are the (hi,lo) pairs of oracle_accumulate. */
int oracle_estimate(const double *sums, uint64_t n_events, double *I, double *sigma)
{
    if (n_events < 2) return ORACLE_EINVAL;
    long double S1 = (long double)sums[0] + (long double)sums[1];
    long double S2 = (long double)sums[2] + (long double)sums[3];
    long double n = (long double)n_events;
    long double mean = S1 / n;
    long double var = (S2 / n - mean * mean) / (n - 1.0L);
    if (!(var > 0.0L)) var = (var != var) ? var : 0.0L;
    *I = (double)mean;
    *sigma = (double)sqrtl(var);
    if (!isfinite(*I) || !isfinite(*sigma)) return ORACLE_ENUMERIC;
    return ORACLE_OK;
}

/* One whole iteration (C2..C7) on a given grid: I, sigma, hist [dim][n_bins] (fp64). */
int oracle_iterate_v(int variant, int dim, int n_bins, const double *edges, uint64_t n_events, uint64_t seed,
                     uint32_t iteration, int integrand_id, const double *params, double *I,
                     double *sigma, double *hist)
{
    double sums[4];
    if (n_events < 2) return ORACLE_EINVAL;
    int rc = oracle_accumulate_v(variant, dim, n_bins, edges, seed, iteration, 0, n_events, integrand_id,
                                 params, sums, hist, NULL);
    if (rc) return rc;
    return oracle_estimate(sums, n_events, I, sigma);
}

int oracle_iterate(int dim, int n_bins, const double *edges, uint64_t n_events, uint64_t seed,
                   uint32_t iteration, int integrand_id, const double *params, double *I,
                   double *sigma, double *hist)
{
    return oracle_iterate_v(0, dim, n_bins, edges, n_events, seed, iteration, integrand_id, params, I, sigma, hist);
}

/* C8  refine one grid from a histogram (classic 1978 Vegas: smooth, normalise, compress with
 * damping alpha, rebin), per dimension, fp64.  A dimension whose smoothed histogram does not
 * have a finite positive sum is left unchanged and ORACLE_ENUMERIC is returned (after all
 * other dimensions have been refined). */
int oracle_refine(int dim, int n_bins, const double *edges, const double *hist, double alpha,
                  double *new_edges)
{
    int rc = check_grid(dim, n_bins, edges);
    if (rc) return rc;
    if (!(alpha >= 0.0)) return ORACLE_EINVAL;
    int status = ORACLE_OK;
    int nb = n_bins;
    double *s = (double *)malloc(sizeof(double) * nb);
    double *m = (double *)malloc(sizeof(double) * nb);
    if (!s || !m) { free(s); free(m); return ORACLE_EINVAL; }
    for (int j = 0; j < dim; ++j) {
        const double *X = edges + (size_t)j * (nb + 1);
        const double *h = hist + (size_t)j * nb;
        double *Y = new_edges + (size_t)j * (nb + 1);
        /* (1) smooth */
        s[0] = (h[0] + h[1]) / 2.0;
        for (int i = 1; i < nb - 1; ++i) s[i] = (h[i - 1] + h[i] + h[i + 1]) / 3.0;
        s[nb - 1] = (h[nb - 2] + h[nb - 1]) / 2.0;
        /* (2) normalise */
        double total = 0.0;
        for (int i = 0; i < nb; ++i) total += s[i];
        if (!(total > 0.0) || !isfinite(total)) {
            for (int i = 0; i <= nb; ++i) Y[i] = X[i];
            status = ORACLE_ENUMERIC;
            continue;
        }
        /* (3) compress: m_i = ((1-p_i)/ln(1/p_i))^alpha */
        double msum = 0.0;
        for (int i = 0; i < nb; ++i) {
            double p = s[i] / total;
            if (p <= 0.0) m[i] = 0.0;
            else if (p >= 1.0) m[i] = 1.0;
            else m[i] = pow((1.0 - p) / log(1.0 / p), alpha);
            msum += m[i];
        }
        /* (4) rebin: equal shares delta of the compressed weight per new bin */
        double delta = msum / (double)nb;
        double C = 0.0;
        int i = 0;
        Y[0] = 0.0;
        for (int k = 1; k < nb; ++k) {
            double t = (double)k * delta;
            while (i < nb - 1 && C + m[i] < t) {
                C += m[i];
                ++i;
            }
            double frac = (m[i] > 0.0) ? (t - C) / m[i] : 0.0;
            if (frac < 0.0) frac = 0.0;
            if (frac > 1.0) frac = 1.0;
            Y[k] = X[i] + frac * (X[i + 1] - X[i]);
        }
        Y[nb] = 1.0;
    }
    free(s);
    free(m);
    return status;
}

/* C9  combine iterations k >= n_skip by inverse-variance weighting:
 * W = sum 1/sigma_k^2; I = sum(I_k/sigma_k^2)/W; sigma = W^-1/2;
 * chi2/dof = sum (I_k - I)^2/sigma_k^2 / (K-1) (0 when K = 1).
 * If any included sigma_k is 0: plain mean of the included I_k, sigma = 0, chi2/dof = 0. */
int oracle_combine(int n_iter, int n_skip, const double *I_k, const double *sigma_k, double *I,
                   double *sigma, double *chi2_dof)
{
    if (n_iter < 1 || n_skip < 0 || n_skip >= n_iter) return ORACLE_EINVAL;
    int K = n_iter - n_skip;
    int any_zero = 0;
    for (int k = n_skip; k < n_iter; ++k)
        if (!(sigma_k[k] > 0.0)) any_zero = 1;
    if (any_zero) {
        long double acc = 0.0L;
        for (int k = n_skip; k < n_iter; ++k) acc += (long double)I_k[k];
        *I = (double)(acc / (long double)K);
        *sigma = 0.0;
        *chi2_dof = 0.0;
        return ORACLE_OK;
    }
    long double W = 0.0L, WI = 0.0L;
    for (int k = n_skip; k < n_iter; ++k) {
        long double w = 1.0L / ((long double)sigma_k[k] * (long double)sigma_k[k]);
        W += w;
        WI += w * (long double)I_k[k];
    }
    long double mean = WI / W;
    long double chi2 = 0.0L;
    for (int k = n_skip; k < n_iter; ++k) {
        long double dev = ((long double)I_k[k] - mean) / (long double)sigma_k[k];
        chi2 += dev * dev;
    }
    *I = (double)mean;
    *sigma = (double)(1.0L / sqrtl(W));
    *chi2_dof = (K > 1) ? (double)(chi2 / (long double)(K - 1)) : 0.0;
    return ORACLE_OK;
}

/* C4  uniform start grid: X[j][i] = (double)i / (double)n_bins. */
void oracle_uniform_edges(int dim, int n_bins, double *edges)
{
    for (int j = 0; j < dim; ++j)
        for (int i = 0; i <= n_bins; ++i)
            edges[(size_t)j * (n_bins + 1) + i] = (double)i / (double)n_bins;
}

/* The whole chain: n_iter iterations of n_events, refine after every iteration (also after the
 * skipped ones), combine k >= n_skip.  edges is in/out ([dim][n_bins+1]); per_iter is
 * [n_iter][2] = (I_k, sigma_k) or NULL; edges_trace is [n_iter][dim][n_bins+1] (the grid each
 * iteration SAMPLED from) or NULL; hist_trace is [n_iter][dim][n_bins] or NULL.
 * alpha < 0 disables refinement (plain importance sampling on a fixed grid). */
int oracle_integrate_v(int variant, int dim, int n_bins, double *edges, int n_iter, int n_skip,
                       uint64_t n_events, uint64_t seed, double alpha, int integrand_id,
                       const double *params, double *I, double *sigma, double *chi2_dof,
                       double *per_iter, double *edges_trace, double *hist_trace)
{
    if (n_iter < 1) return ORACLE_EINVAL;
    size_t ne = (size_t)dim * (n_bins + 1), nh = (size_t)dim * n_bins;
    double *hist = (double *)malloc(sizeof(double) * nh);
    double *next = (double *)malloc(sizeof(double) * ne);
    double *Ik = (double *)malloc(sizeof(double) * n_iter);
    double *sk = (double *)malloc(sizeof(double) * n_iter);
    int status = ORACLE_OK;
    if (!hist || !next || !Ik || !sk) { status = ORACLE_EINVAL; goto done; }
    for (int k = 0; k < n_iter; ++k) {
        if (edges_trace) memcpy(edges_trace + (size_t)k * ne, edges, sizeof(double) * ne);
        int rc = oracle_iterate_v(variant, dim, n_bins, edges, n_events, seed, (uint32_t)k, integrand_id,
                                  params, &Ik[k], &sk[k], hist);
        if (rc) { status = rc; goto done; }
        if (hist_trace) memcpy(hist_trace + (size_t)k * nh, hist, sizeof(double) * nh);
        if (per_iter) { per_iter[2 * k] = Ik[k]; per_iter[2 * k + 1] = sk[k]; }
        if (alpha >= 0.0) {
            rc = oracle_refine(dim, n_bins, edges, hist, alpha, next);
            if (rc == ORACLE_EINVAL) { status = rc; goto done; }
            if (rc == ORACLE_ENUMERIC) status = rc;
            memcpy(edges, next, sizeof(double) * ne);
        }
    }
    {
        int rc = oracle_combine(n_iter, n_skip, Ik, sk, I, sigma, chi2_dof);
        if (rc) status = rc;
    }
done:
    free(hist); free(next); free(Ik); free(sk);
    return status;
}

int oracle_integrate(int dim, int n_bins, double *edges, int n_iter, int n_skip,
                     uint64_t n_events, uint64_t seed, double alpha, int integrand_id,
                     const double *params, double *I, double *sigma, double *chi2_dof,
                     double *per_iter, double *edges_trace, double *hist_trace)
{
    return oracle_integrate_v(0, dim, n_bins, edges, n_iter, n_skip, n_events, seed, alpha, integrand_id, params,
                              I, sigma, chi2_dof, per_iter, edges_trace, hist_trace);
}
