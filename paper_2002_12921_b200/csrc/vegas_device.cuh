// vegas_device.cuh -- device functions shared by the fused iterate kernel (K1) and the parity
// hook (K4): Philox4x32-10, word split, grid map, the built-in integrands, compensated sums.
// sm_100a only.  Readings C1..C11 are those of DESIGN.md; citations are PAPER.md lines.
#pragma once
#ifdef __CUDACC_RTC__
// run-time compilation of a user integrand (vegas_user.cu): NVRTC has no host headers; the fixed-width types
// and the few constants of include/vegas.h the device code uses are restated here
typedef unsigned int uint32_t;
typedef unsigned long long uint64_t;
typedef unsigned long size_t;
#define VEGAS_MAX_DIM 32
#define VEGAS_MAX_PARAMS 160
#define VEGAS_F_CONST 0
#define VEGAS_F_GAUSS 1
#define VEGAS_F_GENZ_PRODUCT_PEAK 2
#ifndef VEGAS_F_GENZ_DISCONTINUOUS
#define VEGAS_F_GENZ_DISCONTINUOUS 5
#endif
#define VEGAS_F_BW_POLY 3
#define VEGAS_F_USER 4
#else
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/vegas.h"
#endif

namespace vegas {

// ------------------------------------------------------------------------------------------
// Integrand parameters as the kernels see them: derived on the host from the user's array
// (vegas_api.cu: derive_params), passed by value as a __grid_constant__ so that every access is a
// constant-bank read with a compile-time offset inside the unrolled dimension loop.
//   GAUSS:  p[0] = (a sqrt(pi))^-d, p[1] = 1/a^2
//   GENZ:   p[2j] = 1/c_j^2, p[2j+1] = w_j
//   BW_POLY: p[0] = s_min, p[1] = s_max - s_min, p[2] = M^2, p[3] = M^2 G^2,
//            p[4 + 5(i-1) + k] = a[i][k]
// ------------------------------------------------------------------------------------------
template <typename T>
struct FParams {
    T p[VEGAS_MAX_PARAMS];
};

// ------------------------------------------------------------------------------------------
// C1: Philox4x32-10.  20 wide multiplies + 20 three-input XORs per block of 4 words; the key
// schedule depends only on the seed, so ptxas keeps it on the uniform datapath.
// ------------------------------------------------------------------------------------------
struct PhiloxKey {
    uint32_t k0[10], k1[10];
};

__device__ __forceinline__ PhiloxKey philox_key_schedule(uint32_t key0, uint32_t key1) {
    PhiloxKey ks;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        ks.k0[r] = key0 + (uint32_t)r * 0x9E3779B9u;
        ks.k1[r] = key1 + (uint32_t)r * 0xBB67AE85u;
    }
    return ks;
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const PhiloxKey& ks, uint32_t (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ ks.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ ks.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ------------------------------------------------------------------------------------------
// C3: split a word into (bin, in-bin offset).  P = word * n_bins exactly; bin = P >> 32.
// fp64: r = (lo + 1/2) 2^-32 exactly, built in the mantissa of a double in [1,2) and shifted down by
//       one exact subtraction (I2F.F64.U32 runs at a quarter of the DADD rate on sm_100).
// fp32 (C11): r32 = ((lo >> 8) + 1/2) 2^-24, within 2^-24 of the fp64 r; the kernel wants
//       r/n_bins because its table stores n_bins*Delta (keeps the Jacobian product in range).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void split_word(uint32_t word, uint32_t n_bins, uint32_t& bin, uint32_t& lo) {
    const uint64_t P = (uint64_t)word * n_bins;
    bin = (uint32_t)(P >> 32);
    lo = (uint32_t)P;
}

__device__ __forceinline__ double offset_f64(uint32_t lo) {
    const double m = __hiloint2double((int)(0x3FF00000u | (lo >> 12)), (int)((lo << 20) | 0x80000u));
    return m - 1.0;
}

__device__ __forceinline__ float offset_f32_scaled(uint32_t lo, float inv_nb_2m24, float inv_nb_2m25) {
    return fmaf((float)(lo >> 8), inv_nb_2m24, inv_nb_2m25);
}

// ------------------------------------------------------------------------------------------
// C5: the built-in integrands in streaming form: begin(), one dim(j, x) call per dimension in
// increasing j, finish() -> f(x).  Nothing of x is kept.
// ------------------------------------------------------------------------------------------
template <typename T> __device__ __forceinline__ T t_exp(T x);
template <> __device__ __forceinline__ double t_exp<double>(double x) { return exp(x); }
template <> __device__ __forceinline__ float t_exp<float>(float x) { return expf(x); }
template <typename T> __device__ __forceinline__ T t_fma(T a, T b, T c);
template <> __device__ __forceinline__ double t_fma<double>(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float t_fma<float>(float a, float b, float c) { return fmaf(a, b, c); }

// exp for the fast path's Gaussian: k = rint(x log2 e) by the 2^52+2^51 shift, r = x - k ln2 in two pieces,
// Taylor series to r^13 on |r| <= ln2/2 (truncation 4e-18 relative) evaluated by Estrin's scheme (depth 4 instead
// of 13 dependent DFMAs: a dependent DFMA issues every ~14 clk, and this tail is serial in every event) or by
// Horner's (template flag), 2^k added into the exponent field.  The coefficients sit in the constant bank, so every DFMA takes its constant as an
// operand: 20 fp64 instructions and 3 integer ones, against ~45 (half of them constant moves) for the library
// routine.  Outside |x| < 700 (results near the ends of the fp64 range) it defers to the library's exp.
static __constant__ double kExpTaylor[14] = {
    1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880, 1.0 / 3628800,
    1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0};

template <bool ESTRIN> __device__ __forceinline__ double exp_fast(double x) {
    if (!(fabs(x) < 700.0)) return exp(x);
    const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
    const int k = __double2loint(t);
    const double kd = t - 6755399441055744.0;
    double r = fma(kd, -6.93147180369123816490e-01, x);      // ln2 high part: 21 trailing zero bits, k ln2_hi exact
    r = fma(kd, -1.90821492927058770002e-10, r);
    if (!ESTRIN) {                 // Horner: 2 instructions and ~8 registers fewer; measured faster for d > 12
        double h = kExpTaylor[13];
#pragma unroll
        for (int n = 12; n >= 0; --n) h = fma(h, r, kExpTaylor[n]);
        return __hiloint2double(__double2hiint(h) + (k << 20), __double2loint(h));
    }
    const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;
    const double a0 = fma(kExpTaylor[1], r, kExpTaylor[0]), a1 = fma(kExpTaylor[3], r, kExpTaylor[2]);
    const double a2 = fma(kExpTaylor[5], r, kExpTaylor[4]), a3 = fma(kExpTaylor[7], r, kExpTaylor[6]);
    const double a4 = fma(kExpTaylor[9], r, kExpTaylor[8]), a5 = fma(kExpTaylor[11], r, kExpTaylor[10]);
    const double a6 = fma(kExpTaylor[13], r, kExpTaylor[12]);
    const double b0 = fma(a1, r2, a0), b1 = fma(a3, r2, a2), b2 = fma(a5, r2, a4);
    const double d0 = fma(b1, r4, b0), d1 = fma(a6, r4, b2);
    const double p = fma(d1, r8, d0);
    return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}
template <typename T, bool ESTRIN> struct ExpFast;
template <bool ESTRIN> struct ExpFast<double, ESTRIN> { static __device__ __forceinline__ double f(double x) { return exp_fast<ESTRIN>(x); } };
template <bool ESTRIN> struct ExpFast<float, ESTRIN> { static __device__ __forceinline__ float f(float x) { return expf(x); } };

template <int FID, typename T>
struct Integrand;

template <typename T>
struct Integrand<VEGAS_F_CONST, T> {
    __device__ __forceinline__ void begin() {}
    __device__ __forceinline__ void dim(int, T, const FParams<T>&) {}
    __device__ __forceinline__ T finish(const FParams<T>&) const { return (T)1; }
};

template <typename T>
struct Integrand<VEGAS_F_GAUSS, T> {   // PAPER.md:65 Eq.(1)
    T s;
    __device__ __forceinline__ void begin() { s = (T)0; }
    __device__ __forceinline__ void dim(int, T x, const FParams<T>&) {
        const T t = x - (T)0.5;
        s = t_fma(t, t, s);
    }
    __device__ __forceinline__ T finish(const FParams<T>& fp) const { return fp.p[0] * t_exp<T>(-s * fp.p[1]); }
};

template <typename T>
struct Integrand<VEGAS_F_GENZ_PRODUCT_PEAK, T> {   // PAPER.md:74 Eq.(3), N = 1
    T prod;
    __device__ __forceinline__ void begin() { prod = (T)1; }
    __device__ __forceinline__ void dim(int j, T x, const FParams<T>& fp) {
        const T t = x - fp.p[2 * j + 1];
        prod *= t_fma(t, t, fp.p[2 * j]);
    }
    __device__ __forceinline__ T finish(const FParams<T>&) const { return (T)1 / prod; }
};

template <typename T>
struct Integrand<VEGAS_F_GENZ_DISCONTINUOUS, T> {   // served through the affine variable (IntegrandU) by both kernels
    __device__ __forceinline__ void begin() {}
    __device__ __forceinline__ void dim(int, T, const FParams<T>&) {}
    __device__ __forceinline__ T finish(const FParams<T>&) const { return (T)0; }
};

template <typename T>
struct Integrand<VEGAS_F_BW_POLY, T> {   // BASELINE.json:configs[4], readings R11, R12
    T bw, poly;
    __device__ __forceinline__ void begin() { bw = (T)0; poly = (T)0; }
    __device__ __forceinline__ void dim(int j, T x, const FParams<T>& fp) {
        if (j == 0) {
            const T ds = t_fma(x, fp.p[1], fp.p[0]) - fp.p[2];        // s - M^2
            bw = fp.p[3] / t_fma(ds, ds, fp.p[3]);
        } else {
            const T* a = &fp.p[4 + 5 * (j - 1)];
            T h = a[4];
            h = t_fma(h, x, a[3]);
            h = t_fma(h, x, a[2]);
            h = t_fma(h, x, a[1]);
            h = t_fma(h, x, a[0]);
            poly += h;
        }
    }
    __device__ __forceinline__ T finish(const FParams<T>&) const { return bw * poly; }
};

// ------------------------------------------------------------------------------------------
// Compensated sums.  Per-thread Kahan accumulators (value s, compensation c; the sum is s - c),
// merged as double-double (hi, lo) pairs, so that S1 and S2 are good to ~1e-30 relative and the
// cancellation in S2/n - I^2 (reading C7) costs nothing even when sigma << I.
// ------------------------------------------------------------------------------------------
struct dd {
    double hi, lo;
};

__device__ __forceinline__ void kahan_add(double& s, double& c, double v) {
    const double y = __dsub_rn(v, c);
    const double t = __dadd_rn(s, y);
    c = __dsub_rn(__dsub_rn(t, s), y);
    s = t;
}

__device__ __forceinline__ dd two_sum(double a, double b) {
    const double s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    const double e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
    return dd{s, e};
}

__device__ __forceinline__ dd fast_two_sum(double a, double b) {   // |a| >= |b|
    const double s = __dadd_rn(a, b);
    return dd{s, __dsub_rn(b, __dsub_rn(s, a))};
}

__device__ __forceinline__ dd dd_add(dd x, dd y) {
    dd s = two_sum(x.hi, y.hi);
    s.lo = __dadd_rn(s.lo, __dadd_rn(x.lo, y.lo));
    return fast_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_neg(dd x) { return dd{-x.hi, -x.lo}; }

__device__ __forceinline__ dd dd_div_d(dd x, double n) {   // x / n
    const double q1 = __ddiv_rn(x.hi, n);
    const double r = __fma_rn(-q1, n, x.hi);                 // exact remainder
    const double q2 = __ddiv_rn(__dadd_rn(r, x.lo), n);
    return fast_two_sum(q1, q2);
}

__device__ __forceinline__ dd dd_sqr(dd x) {
    const double p = __dmul_rn(x.hi, x.hi);
    const double e = __fma_rn(x.hi, x.hi, -p);
    return fast_two_sum(p, __fma_rn(2.0 * x.hi, x.lo, e));
}

__device__ __forceinline__ dd dd_shfl_xor(dd v, int mask) {
    return dd{__shfl_xor_sync(0xffffffffu, v.hi, mask), __shfl_xor_sync(0xffffffffu, v.lo, mask)};
}

__device__ __forceinline__ dd dd_warp_sum(dd v) {
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) v = dd_add(v, dd_shfl_xor(v, m));
    return v;
}

// ------------------------------------------------------------------------------------------
// S5/S6 second level, S7 and S8 as device functions: the stand-alone kernels K2, finalize and K3 (vegas_kernels.cu)
// and the tail that the last CTA of a fused iterate launch runs (vegas_iterate_rot.cuh) call the same code, so an
// iteration gives the same bits whichever way it is finished.
// ------------------------------------------------------------------------------------------

// K2, one of the two double-double sums (i = 0: S1, i = 2: S2) by one warp: lane l adds the partials of CTAs
// l, l+32, ... in that order, then a fixed shuffle tree -- the same association for every run of a launch shape.
// (loads through L2, __ldcg: in the fused tail the rows were written by other CTAs of the same launch)
__device__ __forceinline__ void reduce_dd_sum(const double* partials, int n_parts, int n_tot, int i, int lane, double* totals) {
    dd s{0.0, 0.0};
    for (int p = lane; p < n_parts; p += 32)
        s = dd_add(s, dd{__ldcg(partials + (size_t)p * n_tot + i), __ldcg(partials + (size_t)p * n_tot + i + 1)});
    s = dd_warp_sum(s);
    if (lane == 0) { totals[i] = s.hi; totals[i + 1] = s.lo; }
}

// K2, one slice of a histogram total: the partials of CTAs w, w+8, w+16, ... added in that order (8 loads in flight)
__device__ __forceinline__ double reduce_hist_slice(const double* partials, int n_parts, int n_tot, int i, int w) {
    double h = 0.0;
    int p = w;
    for (; p + 56 < n_parts; p += 64) {
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = __ldcg(partials + (size_t)(p + 8 * k) * n_tot + i);
#pragma unroll
        for (int k = 0; k < 8; ++k) h += v[k];
    }
    for (; p < n_parts; p += 8) h += __ldcg(partials + (size_t)p * n_tot + i);
    return h;
}
constexpr int kReduceSlices = 8;

// S7 (C7): I = S1/n; Var = (S2/n - I^2)/(n-1); sigma = sqrt(max(Var, 0)), in double-double.
// result = { I, sigma, status } (status 0 or VEGAS_ENUMERIC as a double).
__device__ __forceinline__ void finalize_result(const double* totals, double n, double* result) {
    const dd S1 = fast_two_sum(totals[0], totals[1]);
    const dd S2 = fast_two_sum(totals[2], totals[3]);
    const dd mean = dd_div_d(S1, n);
    const dd ex2 = dd_div_d(S2, n);
    const dd diff = dd_add(ex2, dd_neg(dd_sqr(mean)));
    const dd var = dd_div_d(diff, n - 1.0);
    const double v = var.hi + var.lo;
    const double I = mean.hi + mean.lo;
    const double sigma = (v > 0.0) ? sqrt(v) : ((v != v) ? v : 0.0);
    result[0] = I;
    result[1] = sigma;
    result[2] = (isfinite(I) && isfinite(sigma) && isfinite(S2.hi)) ? 0.0 : -3.0 /* VEGAS_ENUMERIC */;
}

// S8 (C8) for one dimension by a group of `gsize` threads (a whole CTA: SYNC = __syncthreads; one warp: SYNC =
// __syncwarp), thread `gi` of the group.  The two running sums that decide where the new edges fall (sum of s_i,
// cumulative sum of m_i) are formed by thread 0 of the group in index order, i.e. in the order the method states them,
// so the walk "advance while C + m_i < t" sees the same doubles whichever thread evaluates it.
// scratch: 4 n_bins + 3 doubles of shared memory for the group.  *status is set to VEGAS_ENUMERIC (-3) if the
// dimension has no finite positive smoothed sum (its grid is left unchanged).
struct SyncCta { __device__ __forceinline__ void operator()() const { __syncthreads(); } };
struct SyncWarp { __device__ __forceinline__ void operator()() const { __syncwarp(); } };
template <class SYNC>
__device__ __forceinline__ void refine_dimension(double* Xg, const double* h, int nb, double alpha,
                                                 int* status, double* scratch, int gi, int gsize, SYNC sync) {
    double* X = scratch;                 // nb + 1
    double* m = X + nb + 1;              // nb
    double* cum = m + nb;                // nb + 1
    double* s = cum + nb + 1;            // nb
    double* total_s = s + nb;            // 1
    for (int i = gi; i < nb; i += gsize) {
        X[i] = Xg[i];
        if (i == 0) X[nb] = Xg[nb];
        double si;
        if (i == 0) si = (h[0] + h[1]) / 2.0;
        else if (i == nb - 1) si = (h[nb - 2] + h[nb - 1]) / 2.0;
        else si = (h[i - 1] + h[i] + h[i + 1]) / 3.0;
        s[i] = si;
    }
    sync();
    if (gi == 0) {
        double t = 0.0;
        for (int k = 0; k < nb; ++k) t += s[k];
        *total_s = t;
    }
    sync();
    const double total = *total_s;
    if (!(total > 0.0) || !isfinite(total)) {
        if (gi == 0) *status = -3 /* VEGAS_ENUMERIC */;
        return;   // whole group: this dimension keeps its grid
    }
    for (int i = gi; i < nb; i += gsize) {
        const double p = s[i] / total;
        double mi;
        if (p <= 0.0) mi = 0.0;
        else if (p >= 1.0) mi = 1.0;
        else mi = pow((1.0 - p) / log(1.0 / p), alpha);
        m[i] = mi;
    }
    sync();
    if (gi == 0) {
        double c = 0.0;
        cum[0] = 0.0;
        for (int k = 0; k < nb; ++k) { c += m[k]; cum[k + 1] = c; }
    }
    sync();
    for (int i = gi; i < nb; i += gsize) {
        if (i >= 1) {
            const double delta = cum[nb] / (double)nb;
            const double t = (double)i * delta;
            int k = 0;
            while (k < nb - 1 && cum[k + 1] < t) ++k;        // cum[k+1] == C + m_k of the sequential walk
            double frac = (m[k] > 0.0) ? (t - cum[k]) / m[k] : 0.0;
            frac = fmin(fmax(frac, 0.0), 1.0);
            Xg[i] = X[k] + frac * (X[k + 1] - X[k]);
        }
    }
    if (gi == 0) { Xg[0] = 0.0; Xg[nb] = 1.0; }
}
__host__ __device__ constexpr size_t refine_scratch_doubles(int n_bins) { return 4 * (size_t)n_bins + 3; }

}  // namespace vegas
