// vegas_iterate_rot.cuh -- K1, "rotated" fast path of the fused iterate kernel (sm_100a).
//
// Same computation as the generic k_iterate (vegas_kernels.cu), for integrands whose dependence on
// x_j goes through a per-dimension affine variable u_j = scale_j (x_j - shift_j)
// (CONST, GAUSS: u = n_bins (x - 1/2); GENZ product peak: u = c_j (x - w_j); Genz discontinuous: u = c_j (x - a_j);
// BW_POLY: u_0 = (s - M^2)/(M Gamma), u_j = x_j; user integrands: u_j = x_j).  Design points, each driven by a counter
// in profiles/ (r01_s2_baseline.md, r01_s2_ubench_hist.md, r02_ubench_pipes.md, r02_k1_steps.md, r02_k1_final.md):
//
//  1. DIM is a compile-time constant: no per-dimension guards, fully unrolled, bins packed one byte
//     per dimension in registers.
//  2. Affine pre-composition: the shared-memory table holds, per (dimension, bin), the pair
//     (A, B) with u = A + B w, where w is the low product word of the split (C3) converted by one
//     I2F (fp64: exact; u = scale (x - shift) with r = (w + 1/2) 2^-32 folded into A and B), the whole
//     Philox word (fp64, more than 8 dimensions: RotSplit<double, true>, no wide multiply in the split) or the
//     top 23 bits of the low product word put into a float mantissa (fp32).  One FMA gives u; x_j itself is never formed,
//     and B is the Jacobian factor up to a per-dimension constant folded into post_scale.
//     No integrand parameter is read inside the event loop.
//  3. Bank rotation.  A Philox block serves 4 dimensions.  The 32 lanes of a warp are split into 4
//     groups gamma = (lane>>1)&3; at sub-step i group gamma works on dimension 4 blk + (gamma ^ i)
//     (its four Philox words are permuted accordingly, 8 SELs per block).  So the lanes of one
//     shared-memory wavefront always touch different dimensions, and the rows
//         table [bin*NBLK + blk] : 128 B = 4 dim-slots x 2 copies x 16 B   (fp32: 4 x 4 x 8 B)
//         hist  [bin*NBLK + blk] : 256 B = 2 half-warps x 4 dim-slots x 4 copies x 8 B
//     (ordered [bin][block]: the block enters every address as a compile-time immediate)
//     are conflict-free whatever bins the lanes drew, with 2 table copies and 8 histogram copies
//     instead of 8 and 32, and no two lanes of a warp ever touch the same histogram word in one
//     instruction.  A last block with 2 (1) dimensions uses 2 (1) groups and 4 (8) table copies in
//     the same row size; with 3 dimensions it uses 4 groups and one idle sub-step.
//  4. Exclusive histogram ownership instead of atomics.  sm_100a has no native fp64 (or fp32, or
//     64-bit integer) shared-memory atomic: atomicAdd(double) is an LDS + DADD + ATOMS.CAST.SPIN + BRA
//     loop that costs 6.4 shared wavefronts and serialises the 20 updates of an event.  Here the CTA
//     (one per SM, sharing one table) holds n_groups histogram copies; the `ring` warps of a group
//     pass a token round a ring (named barriers, bar.sync / bar.arrive on 64 threads, 42 clk per hand-off, for
//     CTAs of up to 16 warps; mbarriers, one per warp and histogram section, for the 24-warp kernels) and only
//     the token holder updates the group's histogram, with plain LDS.64 / DADD / STS.64 (4 wavefronts), the
//     updates of the independent Philox blocks pipelined.  When the shared memory holds one histogram per warp
//     (small dim * n_bins) the ring has length 1 and there is no synchronisation at all.
//  5. One launch per iteration: the chunk loop runs inside the kernel, and the last CTAs to finish reduce the
//     partial rows in K2's fixed association, finalise (S7) and refine the grid (S8): rot_tail.
#pragma once
#include "vegas_device.cuh"
#ifndef __CUDACC_RTC__
#include "vegas_kernels.h"
#endif

namespace vegas {

// ---- integrands in the affine variable u --------------------------------------------------------
// RotCtx<FID, T, NBLK>: what a lane needs about the dimension it handles at (Philox block blk, sub-step i).
// That dimension, 4 blk + (gamma ^ i), is fixed for the whole kernel, so per-dimension integrand parameters
// are picked once, in the prologue, and sit in registers: no select and no parameter read in the event loop.
template <int FID, typename T, int NBLK> struct RotCtx {
    template <class A> __device__ __forceinline__ void init(const A&, int /*dim*/, int /*gamma4*/, int /*gammaL*/) {}
};
// independent accumulator chains per event: 4 for d <= 12; one for larger d, where the 128-register budget of the
// 15-warp CTA is tight and the extra accumulators cost more than the shorter chains give (cfg3: 3.85e10 events/s
// with 1 chain and Horner exp, 3.76e10 with 2 chains, 3.68e10 with 4 chains and Estrin; cfg4: 4.93e10 -> 5.24e10
// and cfg2: 8.03e10 -> 8.10e10 with 4)
// (fp32 product peak and fp32 BW_POLY: always 4, so that no partial product leaves the fp32 range, see their value())
__host__ __device__ constexpr int rot_chains(int dim, int fid = -1, bool fp32 = false) {
    return (fp32 && (fid == VEGAS_F_GENZ_PRODUCT_PEAK || fid == VEGAS_F_BW_POLY || fid == VEGAS_F_USER)) ? 4 : (dim > 12 ? 1 : 4);
}
template <int NCH, typename T> __device__ __forceinline__ T chain_sum(const T (&s)[NCH]) {
    if (NCH == 4) return (s[0] + s[NCH > 1 ? 1 : 0]) + (s[NCH > 2 ? 2 : 0] + s[NCH > 3 ? 3 : 0]);
    if (NCH == 2) return s[0] + s[NCH > 1 ? 1 : 0];
    return s[0];
}
template <int NCH, typename T> __device__ __forceinline__ T chain_prod(const T (&s)[NCH]) {
    if (NCH == 4) return (s[0] * s[NCH > 1 ? 1 : 0]) * (s[NCH > 2 ? 2 : 0] * s[NCH > 3 ? 3 : 0]);
    if (NCH == 2) return s[0] * s[NCH > 1 ? 1 : 0];
    return s[0];
}
template <int FID, typename T, int NCH> struct IntegrandU;

template <typename T, int NCH> struct IntegrandU<VEGAS_F_CONST, T, NCH> {
    template <class C> __device__ __forceinline__ void begin(const C&) {}
    template <class C> __device__ __forceinline__ void dim(T, int, int, const C&) {}
    __device__ __forceinline__ T finish(T, T) const { return (T)1; }
    __device__ __forceinline__ T value(const T (&jac)[NCH], T, T) const { return chain_prod<NCH, T>(jac); }
};
// Every integrand keeps NCH partial accumulators, picked by the sub-step i (NCH independent chains instead of one
// chain of d links: a dependent DFMA issues every ~14 clk on sm_100, r01_s7_ubench_pipes.md), combined in finish().
template <typename T, int NCH> struct IntegrandU<VEGAS_F_GAUSS, T, NCH> {   // PAPER.md:65 Eq.(1); u = n_bins (x - 1/2)
    T s[NCH];
    template <class C> __device__ __forceinline__ void begin(const C&) {
#pragma unroll
        for (int c = 0; c < NCH; ++c) s[c] = (T)0;
    }
    template <class C> __device__ __forceinline__ void dim(T u, int, int i, const C&) {
        s[i & (NCH - 1)] = t_fma(u, u, s[i & (NCH - 1)]);
    }
    // fin0 = 1/(n_bins a)^2.  fp32: fin1 = ln N (the rest of N, a factor 1 +- 2e-6, sits in post_scale), so that
    // f = N exp(-E) leaves the fp32 range where N exp(-E) does, not already where exp(-E) does (34 decades earlier
    // for cfg3's N = 1.07e15).
    __device__ __forceinline__ T finish(T fin0, T fin1) const {
        if (sizeof(T) == 4) return ExpFast<T, (NCH > 1)>::f(t_fma(-chain_sum<NCH, T>(s), fin0, fin1));
        return ExpFast<T, (NCH > 1)>::f(-chain_sum<NCH, T>(s) * fin0);
    }
    __device__ __forceinline__ T value(const T (&jac)[NCH], T fin0, T fin1) const { return finish(fin0, fin1) * chain_prod<NCH, T>(jac); }
};
template <typename T, int NCH> struct IntegrandU<VEGAS_F_GENZ_PRODUCT_PEAK, T, NCH> {   // PAPER.md:74 Eq.(3); u = c_j (x - w_j)
    T prod[NCH];
    template <class C> __device__ __forceinline__ void begin(const C&) {
#pragma unroll
        for (int c = 0; c < NCH; ++c) prod[c] = (T)1;
    }
    template <class C> __device__ __forceinline__ void dim(T u, int, int i, const C&) {
        prod[i & (NCH - 1)] *= t_fma(u, u, (T)1);
    }
    __device__ __forceinline__ T finish(T, T) const { return (T)1 / chain_prod<NCH, T>(prod); }
    // fp32 (C11): f J = prod_j c_j n_bins Delta_j c_j / (1 + u_j^2) is O(I), but prod (1 + u^2) and prod Delta alone
    // leave the fp32 range in many dimensions.  Each of the 4 chains (<= 8 dimensions) is divided on its own and takes
    // a quarter of n_bins^d: fin1 = n_bins^(d/4) (what rounding leaves of n_bins^d / fin1^4 sits in post_scale).
    __device__ __forceinline__ T value(const T (&jac)[NCH], T fin0, T fin1) const {
        if (sizeof(T) == 4 && NCH == 4) {
            T r[NCH];
#pragma unroll
            for (int c = 0; c < NCH; ++c) r[c] = (jac[c] * fin1) / prod[c];
            return chain_prod<NCH, T>(r);
        }
        return finish(fin0, fin1) * chain_prod<NCH, T>(jac);
    }
};
// Genz discontinuous, Eq.(2) as printed (reading R19): u_j = c_j (x_j - a_j), c_j > 0, so that the cut
// x_j <= a_j is u_j <= 0 and sum_j c_j x_j = sum_j u_j + sum_j c_j a_j (fin1).  fp64 only (include/vegas.h).
template <typename T, int NCH> struct IntegrandU<VEGAS_F_GENZ_DISCONTINUOUS, T, NCH> {
    T s[NCH];
    bool cut;
    template <class C> __device__ __forceinline__ void begin(const C&) {
#pragma unroll
        for (int c = 0; c < NCH; ++c) s[c] = (T)0;
        cut = false;
    }
    template <class C> __device__ __forceinline__ void dim(T u, int, int i, const C&) {
        s[i & (NCH - 1)] += u;
        cut = cut || !(u > (T)0);
    }
    __device__ __forceinline__ T finish(T, T fin1) const {
        return cut ? (T)0 : ExpFast<T, (NCH > 1)>::f(chain_sum<NCH, T>(s) + fin1);
    }
    __device__ __forceinline__ T value(const T (&jac)[NCH], T fin0, T fin1) const { return finish(fin0, fin1) * chain_prod<NCH, T>(jac); }
};
// BW_POLY (BASELINE.json:configs[4], readings R11, R12): u_0 = (s(x_0) - M^2)/(M Gamma), u_j = x_j for j >= 1;
// f = [1/(1 + u_0^2)] * [sum_j a_j0 + sum_j u_j (a_j1 + u_j (a_j2 + u_j (a_j3 + u_j a_j4)))].
// The lane that holds dimension 0 at sub-step i of block 0 runs the quartic with zero coefficients and keeps u.
constexpr int kRotBwMaxDim = 8;    // up to here a lane keeps the 4 coefficients of each of its dimensions in registers;
                                   // beyond, it reads them from the kernel arguments (constant bank) by dimension index
constexpr int kRotMaxObsBins = 128; // observable histogram of a user integrand (vegas_set_observable)
constexpr int kRotParams = 5 * VEGAS_MAX_DIM;   // doubles of integrand parameters carried in the kernel arguments
                                                // (BW_POLY: 5 per dimension; USER: VEGAS_USER_MAX_PARAMS = 64 of them)
template <typename T, int NCH> struct IntegrandU<VEGAS_F_BW_POLY, T, NCH> {
    T poly[NCH], u0;
    template <class C> __device__ __forceinline__ void begin(const C& c) {
#pragma unroll
        for (int k = 0; k < NCH; ++k) poly[k] = k ? (T)0 : c.poly0;
        u0 = (T)0;
    }
    template <class C> __device__ __forceinline__ void dim(T u, int blk, int i, const C& c) {
        T a4[4];
        c.coefs(blk, i, a4);
        T h = t_fma(a4[3], u, a4[2]);
        h = t_fma(h, u, a4[1]);
        h = t_fma(h, u, a4[0]);
        poly[i & (NCH - 1)] = t_fma(h, u, poly[i & (NCH - 1)]);
        if (blk == 0 && c.dim0(i)) u0 = u;
    }
    // reciprocal first: it depends on u_0 alone, so it runs beside the polynomial chains; one multiply follows them
    __device__ __forceinline__ T finish(T, T) const { return chain_sum<NCH, T>(poly) * ((T)1 / t_fma(u0, u0, (T)1)); }
    // fp32 (C11): prod Delta_j alone leaves the fp32 range in many dimensions (u_j = x_j: the table carries no
    // n_bins); each of the 4 chains takes a quarter of n_bins^d first: fin1 = n_bins^(d/4), the rest is in post_scale
    __device__ __forceinline__ T value(const T (&jac)[NCH], T fin0, T fin1) const {
        if (sizeof(T) == 4 && NCH == 4) {
            T r[NCH];
#pragma unroll
            for (int c = 0; c < NCH; ++c) r[c] = jac[c] * fin1;
            return finish(fin0, fin1) * chain_prod<NCH, T>(r);
        }
        return finish(fin0, fin1) * chain_prod<NCH, T>(jac);
    }
};

// ---- table entry and u from the low product word ---------------------------------------------------
template <typename T> struct RotEntry;
template <> struct RotEntry<double> {
    using type = double2;
    // u = scale (X_b + Delta r - shift), r = (w + 1/2) 2^-32  ==>  u = A + B' w with
    // B' = scale Delta 2^-32 (exact scaling) and A = scale (X_b - shift) + B'/2.  The Jacobian factor is
    // B' 2^32 / scale; the 2^32 per dimension goes into post_scale (vegas_api.cu: rot_constants).
    // (the generic kernel's form: w is the low word of the split product)
    static __device__ __forceinline__ double2 make(double x0, double x1, double shift, double scale) {
        const double B = (x1 - x0) * scale, A = (x0 - shift) * scale;
        return make_double2(fma(B, 1.1641532182693481e-10, A), B * 2.3283064365386963e-10);   // 2^-33, 2^-32
    }
    static __device__ __forceinline__ double u(double2 e, uint32_t lo) {
        return fma(e.y, (double)lo, e.x);              // I2F.F64.U32 (its own pipe) + DFMA
    }
    static constexpr double kJacUnit = 4294967296.0;   // table B = kJacUnit^-1 * scale * Delta
    // The fast path's form: u as an affine function of the WHOLE Philox word W of the dimension, per bin b.
    // With P = W n_bins, b = P >> 32 and lo = P - b 2^32 (C3), r = (lo + 1/2) 2^-32 = W n_bins 2^-32 - b + 2^-33, so
    //   u = A_b + B_b W,   B_b = scale Delta n_bins 2^-32,   A_b = scale (X_b - shift) + scale Delta (2^-33 - b).
    // The split needs no integer multiply then (IMAD.WIDE.U32 costs 3.4..4.4 issue clocks on sm_100a, a DFMA 1.3..2:
    // profiles/r02_ubench_pipes.md): with Wd = (double)W, t = RZ(Wd n_bins 2^-32 + 2^52) has b = floor(P 2^-32) in its
    // low word -- exactly, the sum is formed exactly before the one rounding towards zero -- and u = fma(B_b, Wd, A_b).
    // A_b + B_b W cancels Delta b, so u carries an absolute error of ~1.5e-16 scale (x_j within ~3e-16 absolute of
    // the plain map instead of 1 ulp; reading R21); the Jacobian factor B_b is a product of exact values.
    static __device__ __forceinline__ double2 make_w(double x0, double x1, double shift, double scale, int b, int n_bins) {
        const double B = (x1 - x0) * scale, A = (x0 - shift) * scale;
        return make_double2(fma(B, 1.1641532182693481e-10 - (double)b, A), B * ((double)n_bins * 2.3283064365386963e-10));
    }
};
template <> struct RotEntry<float> {
    using type = float2;
    static __device__ __forceinline__ float2 make(double x0, double x1, double shift, double scale) {
        const double B = (x1 - x0) * scale, A = (x0 - shift) * scale;
        // m = 1 + k 2^-23 with k = lo >> 9; the half-step 2^-24 centres r within 2^-24 of C3's r (C11)
        return make_float2((float)(A - B + B * 5.9604644775390625e-08), (float)B);
    }
    static __device__ __forceinline__ float u(float2 e, uint32_t lo) {
        const float m = __uint_as_float(__funnelshift_r(lo, 0x7Fu, 9));
        return fmaf(e.y, m, e.x);
    }
    static constexpr double kJacUnit = 1.0;
};

// C3 + C4 on the fast path: word -> (bin, operand of the table entry's affine map), and the entry itself.  Bins are
// bit-exact in both forms.  WORD (fp64 only): the entry is affine in the whole word (RotEntry<double>::make_w).
// It pays where the kernel is bound by its instruction stream (more than 8 dimensions: cfg3 +1 %, cfg4 +5 %); the
// small shapes are latency-bound and lose (cfg5 -7 %), they keep the integer split.
#ifndef VEGAS_ROT_WORD_MIN_DIM
#define VEGAS_ROT_WORD_MIN_DIM 9
#endif
__host__ __device__ constexpr bool rot_word_map(int precision_bits, int dim) {
    return precision_bits == 64 && dim >= VEGAS_ROT_WORD_MIN_DIM;
}
template <typename T, bool WORD> struct RotSplit;
template <> struct RotSplit<double, true> {
    using arg = double;                                  // the word itself as a double (I2F.F64.U32, exact)
    static __device__ __forceinline__ void split(uint32_t w, uint32_t, double nb_2m32, uint32_t& b, double& o) {
        o = (double)w;
        b = (uint32_t)__double2loint(__fma_rz(o, nb_2m32, 4503599627370496.0));       // 2^52 + floor(w n_bins 2^-32)
    }
    static __device__ __forceinline__ double u(double2 e, double o) { return fma(e.y, o, e.x); }
    static __device__ __forceinline__ double2 make(double x0, double x1, double shift, double scale, int b, int nb) {
        return RotEntry<double>::make_w(x0, x1, shift, scale, b, nb);
    }
};
template <typename T> struct RotSplit<T, false> {
    using arg = uint32_t;                                // the low word of the product (fp32, C11: its top 23 bits are used)
    static __device__ __forceinline__ void split(uint32_t w, uint32_t nb, double, uint32_t& b, uint32_t& o) {
        split_word(w, nb, b, o);
    }
    static __device__ __forceinline__ T u(typename RotEntry<T>::type e, uint32_t o) { return RotEntry<T>::u(e, o); }
    static __device__ __forceinline__ typename RotEntry<T>::type make(double x0, double x1, double shift, double scale, int, int) {
        return RotEntry<T>::make(x0, x1, shift, scale);
    }
};

// ---- variants of the sampling map (readings C3', C4'; fp64, built-in integrands) ------
// VAR 0: the method (C2, C3, C4).
// VAR 1 (VEGAS_VARIANT_U53, C3'): 53-bit uniforms, two Philox words per draw: one Philox block serves two dimensions
//        (counter word 0 = j >> 1), U = hi 2^21 + (lo >> 11), P = U n_bins, b = P >> 53, r = (P mod 2^53) 2^-53.
//        Table entry (A, B) = (scale (X_b - shift), scale Delta 2^-53), u = A + B (double)(P mod 2^53).
// VAR 2 (VEGAS_VARIANT_Q32, C4'): the table holds the per-bin pair (X_b, Delta_b) rounded to fp32 (8 bytes per entry,
//        half the table read of VAR 0); x = X~_b + Delta~_b r in fp64, u = scale (x - shift), J = prod n_bins Delta~_b.
constexpr int kVarU53 = 1, kVarQ32 = 2;
__host__ __device__ constexpr int rot_jac_bits(int precision_bits, int var) {     // table B = scale Delta 2^-bits
    return precision_bits != 64 ? 0 : (var == kVarU53 ? 53 : (var == kVarQ32 ? 0 : 32));
}
template <typename T, int VAR> struct RotTableEntry { using type = typename RotEntry<T>::type; };
template <> struct RotTableEntry<double, kVarQ32> { using type = float2; };
struct RotVarU53 {
    static __device__ __forceinline__ double2 make(double x0, double x1, double shift, double scale) {
        return make_double2((x0 - shift) * scale, ((x1 - x0) * scale) * 1.1102230246251565e-16);      // 2^-53
    }
    static __device__ __forceinline__ void split(uint64_t U, uint32_t nb, uint32_t& b, double& o) {
        const uint64_t P = U * (uint64_t)nb;                      // < 2^61
        b = (uint32_t)(P >> 53);
        o = (double)(P & 0x1FFFFFFFFFFFFFull);                    // exact: 53 bits
    }
};
struct RotVarQ32 {
    static __device__ __forceinline__ float2 make(double x0, double x1) { return make_float2((float)x0, (float)(x1 - x0)); }
};
// w'[i] = w[gamma ^ i] for the G lane groups of a block (two conditional swaps, SELs)
template <int G, typename W>
__device__ __forceinline__ void rot_permute(W (&w)[4], int gamma) {
    if (G == 4) {
        const bool g1 = gamma & 1, g2 = gamma & 2;
        const W t0 = g1 ? w[1] : w[0], t1 = g1 ? w[0] : w[1], t2 = g1 ? w[3] : w[2], t3 = g1 ? w[2] : w[3];
        w[0] = g2 ? t2 : t0; w[1] = g2 ? t3 : t1; w[2] = g2 ? t0 : t2; w[3] = g2 ? t1 : t3;
    } else if (G == 2) {
        const bool g1 = gamma & 1;
        const W t0 = g1 ? w[1] : w[0], t1 = g1 ? w[0] : w[1];
        w[0] = t0; w[1] = t1;
    }
}

// 32-bit shared-window addressing: one register per address, no generic-to-shared conversion
template <typename T2> __device__ __forceinline__ T2 lds_entry(uint32_t addr);
template <> __device__ __forceinline__ double2 lds_entry<double2>(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
template <> __device__ __forceinline__ float2 lds_entry<float2>(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ double lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_f64(uint32_t addr, double v) {
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
// Token passing between the warps that share a histogram copy: one mbarrier (arrival count 1) per warp and section
// in shared memory.  The holder's predecessor arrives (release), the waiting warp spins on try_wait (acquire; the
// hardware suspends the warp for a bounded time per attempt, so a waiting warp takes no issue slots to speak of).
// Measured on B200 (profiles/r02_ubench_pipes.md, token rings): 113..124 clk per hand-off against 42 for
// bar.sync/bar.arrive, but the 16 named barriers of a CTA cap a ring scheme at 15 warps, and more warps are worth more
// than the 70 clk (cfg3: 24 warps 4.35e10 events/s, 21 warps 3.84e10; the ring itself is not what cfg3 waits for:
// with a private copy per warp and no tokens at all it runs 4.31e10).
__device__ __forceinline__ void token_init(uint32_t bar) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
}
// try_wait returns after ~12 clk on sm_100a whether or not the phase has completed (a suspend-time hint, nanosleep
// between attempts, or an L2 round trip between attempts all measured the same or slower, round-2 experiments),
// so this is a spin; a waiting warp issues ~3 instructions per 12 clk.
__device__ __forceinline__ void token_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "TOK_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra TOK_WAIT_%=;\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// named barriers 1..15 on 64 threads (rings of up to 15 warps): the waiting warp syncs, the signalling warp arrives
__device__ __forceinline__ void token_wait_named(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void token_pass_named(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void token_pass(uint32_t bar) {          // one lane, after __syncwarp()
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

struct RotArgs {
    const double* edges;            // device, [DIM][n_bins+1]
    double* partials;               // device, [gridDim.x][4 + DIM*n_bins]
    unsigned long long first_event, count;
    unsigned long long chunk;       // events per chunk inside this launch (0 = one chunk): the grid finishes a chunk before
                                    // it starts the next, per-thread sums are folded into double-double at chunk ends
    uint32_t iteration;
    uint32_t k0[10], k1[10];        // Philox key schedule (C1), built on the host: LOP3 reads it from the constant bank
    int n_bins;
    int n_groups, ring;             // histogram copies in the CTA; warps per copy (blockDim = 32 n_groups ring)
    double post_scale;              // v = f_u * jac * post_scale
    double jac_init;                // start value of the running Jacobian product (a power of two, see RotEntry)
    double fin0, fin1;              // integrand finish constants (IntegrandU::finish / value)
    double shift[VEGAS_MAX_DIM], scale[VEGAS_MAX_DIM];
    // The iteration as ONE launch (vegas_iterate / vegas_integrate when the whole iteration fits one launch):
    int overwrite;                  // 1: first launch of an iteration: the CTA's partial row is overwritten, not added to
    int tail;                       // 1: the last CTA to finish reduces the partials (K2), finalises (S7) and, if
                                    //    tail_alpha >= 0, refines the grid (S8) -- same device code as the stand-alone kernels
    double tail_n, tail_alpha;      // events of the whole iteration; damping exponent (< 0: no refinement)
    double* totals;                 // device, [4 + DIM*n_bins]
    double* result;                 // device, { I, sigma, status } of this iteration
    int* status;                    // device, refinement status word
    double* slices;                 // device, [8][DIM*n_bins]: K2's slice sums
    unsigned int* counter;          // device, 8 + 1 CTAs-done tickets (0 before the launch, reset by the last CTA)
    unsigned int tail_smem_doubles; // doubles of dynamic shared memory the launch has (scratch of the refinement)
    int pdl;                        // host side: launch with programmatic stream serialisation (the previous launch in
                                    // the stream is a chunk of the same accumulate call); the kernel does not read it
    double* obs;                    // USER with an observable: device, [n_obs] sums of v per observable bin, or NULL
    int n_obs;                      // 0 = no observable histogram
    double obs_lo, obs_inv_width;   // bin k = floor((O - obs_lo) * obs_inv_width)
    double fpar[kRotParams];        // BW_POLY: a[j][k] at fpar[5 j + k], j = 1..dim-1 (row 0 unused); USER: the caller's array
};

template <typename T, int NBLK> struct RotCtx<VEGAS_F_BW_POLY, T, NBLK> {
    static constexpr bool kRegs = NBLK <= kRotBwMaxDim / 4;
    T a[kRegs ? NBLK : 1][4][4];    // a_j1..a_j4 of the lane's dimension at (blk, i); zero for dimension 0 / no dimension
    bool is0[4];                    // the lane holds dimension 0 at sub-step i of block 0
    T poly0;                        // sum_j a_j0
    uint32_t cbase;                 // more than 8 dimensions: shared-window address of the coefficient rows [dim][4]
                                    // (32 bytes per dimension; the 4 lane groups of a warp read 4 consecutive rows: one
                                    // conflict-free wavefront per LDS.128; reading them from the constant bank by a
                                    // lane-dependent index measured 2x slower than the generic kernel's whole event)
    const double* p;                // the same rows in the kernel arguments (RotArgs::fpar; row 0 is zero): K4's view
    int gamma4, gammaL, nblk;
    template <class A> __device__ __forceinline__ void init(const A& r, int dim, int g4, int gL) {
        nblk = (dim + 3) / 4;
        gamma4 = g4; gammaL = gL; p = r.fpar; cbase = 0;
        T c0 = (T)0;
        for (int j = 1; j < dim; ++j) c0 += (T)r.fpar[5 * j];
        poly0 = c0;
#pragma unroll
        for (int blk = 0; blk < (kRegs ? NBLK : 1); ++blk)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int j = 4 * blk + ((blk == nblk - 1 ? gammaL : gamma4) ^ i);
                const bool poly_dim = blk < nblk && j >= 1 && j < dim;
#pragma unroll
                for (int k = 0; k < 4; ++k) a[blk][i][k] = poly_dim ? (T)r.fpar[5 * j + 1 + k] : (T)0;
                if (blk == 0) is0[i] = (j == 0);
            }
    }
    __device__ __forceinline__ void coefs(int blk, int i, T (&out)[4]) const {
        if (kRegs) {
#pragma unroll
            for (int k = 0; k < 4; ++k) out[k] = a[kRegs ? blk : 0][i][k];
            return;
        }
        const int j = 4 * blk + ((blk == nblk - 1 ? gammaL : gamma4) ^ i);
        if (cbase) {
            const double2 lo = lds_entry<double2>(cbase + 32u * (uint32_t)j), hi = lds_entry<double2>(cbase + 32u * (uint32_t)j + 16u);
            out[0] = (T)lo.x; out[1] = (T)lo.y; out[2] = (T)hi.x; out[3] = (T)hi.y;
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) out[k] = (T)p[5 * j + 1 + k];
        }
    }
    __device__ __forceinline__ bool dim0(int i) const { return is0[i]; }
};

#ifdef VEGAS_USER_INTEGRAND
// A user-supplied integrand compiled at run time (vegas_user.cu): the caller's
// source defines `struct vegas_user_integrand` in streaming form (include/vegas.h: vegas_set_user_integrand);
// it sees x_j itself (scale 1, shift 0) and the index j of the dimension this lane holds at (blk, i).
template <typename T, int NBLK> struct RotCtx<VEGAS_F_USER, T, NBLK> {
    const double* p;
    int gamma4, gammaL, nblk, dim;
    template <class A> __device__ __forceinline__ void init(const A& r, int d, int g4, int gL) {
        p = r.fpar; gamma4 = g4; gammaL = gL; nblk = (d + 3) / 4; dim = d;
    }
};
template <class U> struct user_has_observable {
    template <class V> static __device__ char test(decltype(&V::observable));
    template <class V> static __device__ long test(...);
    static constexpr bool value = sizeof(test<U>(0)) == sizeof(char);
};
template <typename T, int NCH> struct IntegrandU<VEGAS_F_USER, T, NCH> {
    static constexpr bool kObservable = user_has_observable<vegas_user_integrand>::value;
    vegas_user_integrand f;
    __device__ __forceinline__ double observable() {
        if constexpr (kObservable) return f.observable(p);
        else return 0.0;
    }
    const double* p;
    template <class C> __device__ __forceinline__ void begin(const C& c) { p = c.p; f.begin(c.dim, p); }
    template <class C> __device__ __forceinline__ void dim(T u, int blk, int i, const C& c) {
        f.dim(4 * blk + ((blk == c.nblk - 1 ? c.gammaL : c.gamma4) ^ i), (double)u, p);
    }
    __device__ __forceinline__ T finish(T, T) { return (T)f.finish(p); }
    // fp32 (C11): the sampling map, J and v = f J in fp32 around the user's f (evaluated in the user's own types from
    // x widened to double, then rounded to fp32); the four partial Jacobian chains take a quarter of n_bins^d each
    __device__ __forceinline__ T value(const T (&jac)[NCH], T fin0, T fin1) {
        if (sizeof(T) == 4 && NCH == 4) {
            T r[NCH];
#pragma unroll
            for (int c = 0; c < NCH; ++c) r[c] = jac[c] * fin1;
            return finish(fin0, fin1) * chain_prod<NCH, T>(r);
        }
        return finish(fin0, fin1) * chain_prod<NCH, T>(jac);
    }
};
#endif

// One CTA per SM.  Warps per CTA (= __launch_bounds__, i.e. the register budget ptxas works to):
//  * 4 or 5 Philox blocks (dim >= 13): 24 warps at <= 85 registers.  ptxas fits the event loop of every instantiation
//    into 72..80 registers without spills, and the per-event latencies (10 dependent Philox rounds, the exp tail, the
//    histogram round trips) want more warps than the 15 the named-barrier ring allows: cfg3 3.98e10 -> 4.17e10
//    events/s (profiles/r02_k1_steps.md; 27, 30 and 32 warps measured slower again).  Tokens are mbarriers.
//  * up to 3 Philox blocks: 16 warps at <= 128 registers, tokens over named barriers (42 clk per hand-off against 78):
//    most of these shapes give every warp or every other warp its own histogram copy, and measured 3..15 % faster
//    this way (cfg1, cfg2, cfg5).
//  * BW_POLY keeps 4 coefficients per dimension per lane in registers, and a user integrand's register needs are
//    unknown: 12 warps, up to 168 registers.
#ifndef VEGAS_ROT_BW_WARPS
#define VEGAS_ROT_BW_WARPS 12
#endif
#ifndef VEGAS_ROT_WIDE_WARPS
#define VEGAS_ROT_WIDE_WARPS 24
#endif
#ifndef VEGAS_ROT_WIDE_MIN_DIM
#define VEGAS_ROT_WIDE_MIN_DIM 13
#endif
__host__ __device__ constexpr int rot_max_warps(int fid, int dim) {
    return (fid == VEGAS_F_USER || (fid == VEGAS_F_BW_POLY && dim <= kRotBwMaxDim && VEGAS_ROT_BW_WARPS == 12))
               ? 12 : (dim >= VEGAS_ROT_WIDE_MIN_DIM ? VEGAS_ROT_WIDE_WARPS : 16);
}
__host__ __device__ constexpr int rot_max_threads(int fid, int dim) { return 32 * rot_max_warps(fid, dim); }
__host__ __device__ constexpr bool rot_mbar_tokens(int fid, int dim) { return rot_max_warps(fid, dim) > 16; }
constexpr int kRotMaxNamedRingWarps = 15;   // named barriers 1..15 carry the tokens (barrier 0 is __syncthreads)
constexpr int kRotNamedDefaultWarps = 12;
// Sections of a histogram copy: the rows of different Philox blocks are disjoint, so a copy shared by a ring of warps
// is guarded by one token per section (a run of blocks) and the ring is pipelined: while one warp updates the rows of
// blocks 3..4 the next already updates those of blocks 0..2.  Needs one token per warp and section: mbarriers only.
#ifndef VEGAS_ROT_NSEC
#define VEGAS_ROT_NSEC 2
#endif
__host__ __device__ constexpr int rot_sections(int fid, int dim) {
    return !rot_mbar_tokens(fid, dim) ? 1 : ((dim + 3) / 4 < VEGAS_ROT_NSEC ? (dim + 3) / 4 : VEGAS_ROT_NSEC);
}
// Two events per token hold (template parameter PAIR of the kernel, picked at launch when warps share a histogram
// copy): every shape of up to 3 Philox blocks, whose register budget has room for a second set of histogram
// addresses.  It pays most where large tables leave few copies (cfg4: 2 copies, 7 warps each: 5.45e10 -> 5.53e10
// events/s, barrier stalls per issue 3.97 -> 2.53) and 1..2 % on the short rings of the small shapes (cfg2, cfg5:
// two independent events in flight per thread); profiles/r02_k1_steps.md.  A kernel of its own because the second
// loop in the same kernel cost the shapes without rings 5 %.
#ifndef VEGAS_ROT_PAIR_MIN_DIM
#define VEGAS_ROT_PAIR_MIN_DIM 2
#endif
__host__ __device__ constexpr bool rot_pair_hold(int fid, int dim, int var = 0) {
    return fid != VEGAS_F_USER && var == 0 && dim >= VEGAS_ROT_PAIR_MIN_DIM && dim <= 12;
}
__host__ __device__ constexpr int rot_section_begin(int nblk, int nsec, int s) { return (s * nblk + nsec - 1) / nsec; }
constexpr int kRotMaxSections = 8;
constexpr int kRotScratchWarps = 32;   // sizing of the per-warp scratch (reduction slots, tokens): any CTA has <= 32 warps
__host__ __device__ constexpr int rot_groups(int r) { return r >= 3 ? 4 : r; }   // dims in block -> lane groups

// byte offset of (slot 0, this lane's copy) inside a table row, for a block with G lane groups;
// the offset for slot s is this value ^ (s << (7 - log2 G)).  ENTRY = sizeof(table entry) (16 or 8).
template <int G, int ENTRY>
__device__ __forceinline__ uint32_t rot_table_off0(int lane) {
    const int p = lane & 7, b3 = (lane >> 3) & 1;
    constexpr int LG = (G == 4) ? 2 : (G == 2) ? 1 : 0;
    const int gamma = p >> (3 - LG), tc = p & ((8 >> LG) - 1);
    if (ENTRY == 16) return (uint32_t)(gamma * (128 >> LG) + tc * 16);
    return (uint32_t)(gamma * (128 >> LG) + (tc + (8 >> LG) * b3) * 8);     // 8-byte entries: half-warp phases
}
template <int G>
__device__ __forceinline__ uint32_t rot_hist_off0(int lane) {
    const int p = lane & 7, b3 = (lane >> 3) & 1, b4 = lane >> 4;
    constexpr int LG = (G == 4) ? 2 : (G == 2) ? 1 : 0;
    const int gamma = p >> (3 - LG), tc = p & ((8 >> LG) - 1);
    return (uint32_t)(b4 * 128 + gamma * (128 >> LG) + (tc + (8 >> LG) * b3) * 8);
}
template <int G>
__device__ __forceinline__ int rot_gamma(int lane) {
    constexpr int LG = (G == 4) ? 2 : (G == 2) ? 1 : 0;
    return (lane & 7) >> (3 - LG);
}

// per-thread constants of the event loop.  Addresses are 32-bit shared-window addresses; rows are ordered
// [bin][Philox block], so the block enters every address as a compile-time immediate:
//   table entry of (blk, bin, sub-step i):  taddr + 128 blk,  taddr = bin (128 NBLK) + tx[i]   (tx includes the base)
//   histogram word of the same:             haddr + 256 blk,  haddr = 2 taddr + hc[i]
// one multiply-add and one three-input add per dimension, no per-block base to add.
template <typename T, int DIM>
struct RotLane {
    static constexpr int NBLK = (DIM + 3) / 4;
    static constexpr int R = DIM - 4 * (NBLK - 1);               // dimensions in the last block, 1..4
    static constexpr int GL = rot_groups(R);
    uint32_t tbase;
    uint32_t tx4[4], txL[4];      // full blocks / last block: table base + row offset of sub-step i (lane-dependent)
    uint32_t hc4[4], hcL[4];      // haddr - 2 taddr
    int gamma4, gammaL;
};

// C1 with the key schedule taken from the kernel arguments
__device__ __forceinline__ void philox4x32_10_args(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                   const RotArgs& a, uint32_t (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ a.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ a.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// S1..S5 for one event: Philox -> split -> table -> u -> integrand; returns v = f J and leaves the
// histogram address of every (block, sub-step) in haddr (one LEA from the table address, outside the critical section).
template <int FID, typename T, int DIM, int VAR>
__device__ __forceinline__ double rot_event(const RotArgs& a, const RotLane<T, DIM>& L,
                                            const RotCtx<FID, T, (DIM + 3) / 4>& ctx, uint32_t e_lo, uint32_t e_hi,
                                            bool live, T fin0, T fin1, uint32_t (&haddr)[(DIM + 3) / 4][4], double& obs_val) {
    using SP = RotSplit<T, rot_word_map(8 * (int)sizeof(T), DIM) && VAR == 0>;
    using T2 = typename RotTableEntry<T, VAR>::type;
    static_assert(VAR == 0 || sizeof(T) == 8, "the variants are fp64 modes");
    constexpr int NBLK = RotLane<T, DIM>::NBLK, R = RotLane<T, DIM>::R, GL = RotLane<T, DIM>::GL;
    const int nb = a.n_bins;
    const double nb_2m32 = (double)nb * 2.3283064365386963e-10;
    constexpr int NCH = rot_chains(DIM, FID, sizeof(T) == 4);
    IntegrandU<FID, T, NCH> f;
    f.begin(ctx);
    T jac[NCH];                                          // partial Jacobian products (see IntegrandU)
#pragma unroll
    for (int c = 0; c < NCH; ++c) jac[c] = c ? (T)1 : (T)a.jac_init;
#pragma unroll
    for (int blk = 0; blk < NBLK; ++blk) {
        const bool last = (blk == NBLK - 1);
        const int G = last ? GL : 4;
        const int NSUB = last ? ((R == 3) ? 4 : R) : 4;             // sub-steps of this block
        const int gamma = last ? L.gammaL : L.gamma4;
        uint32_t w[4];
        uint64_t U[4];
        (void)U;
        (void)w;
        if constexpr (VAR == kVarU53) {
            // C3': Philox block 2 blk serves dimensions 4 blk, 4 blk + 1; block 2 blk + 1 the next two
            const int dims_here = last ? R : 4;
            uint32_t wa[4], wb[4] = {0u, 0u, 0u, 0u};
            philox4x32_10_args((uint32_t)(2 * blk), a.iteration, e_lo, e_hi, a, wa);
            if (dims_here > 2) philox4x32_10_args((uint32_t)(2 * blk + 1), a.iteration, e_lo, e_hi, a, wb);
            U[0] = ((uint64_t)wa[0] << 21) | (wa[1] >> 11);
            U[1] = ((uint64_t)wa[2] << 21) | (wa[3] >> 11);
            U[2] = ((uint64_t)wb[0] << 21) | (wb[1] >> 11);
            U[3] = ((uint64_t)wb[2] << 21) | (wb[3] >> 11);
            if (G == 4) rot_permute<4>(U, gamma);
            else if (G == 2) rot_permute<2>(U, gamma);
        } else {
            philox4x32_10_args((uint32_t)blk, a.iteration, e_lo, e_hi, a, w);
            if (G == 4) rot_permute<4>(w, gamma);
            else if (G == 2) rot_permute<2>(w, gamma);
        }
        // the block's table reads are issued together, then consumed (their latency overlaps)
        typename SP::arg lo[4];
        double lo53[4];
        (void)lo53;
        T2 ent[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            haddr[blk][i] = 0;
            if (i < NSUB) {
                const bool active = !(last && R == 3) || ((gamma ^ i) < 3);
                uint32_t b = 0;
                lo[i] = 0;
                lo53[i] = 0.0;
                ent[i] = T2{};
                if (active) {
                    if constexpr (VAR == kVarU53) RotVarU53::split(U[i], (uint32_t)nb, b, lo53[i]);
                    else SP::split(w[i], (uint32_t)nb, nb_2m32, b, lo[i]);
                    // one multiply-add (written in C the compiler turns it into shifts and masks of the split product)
                    uint32_t taddr;
                    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(taddr) : "r"(b), "n"(NBLK * 128), "r"(last ? L.txL[i] : L.tx4[i]));
                    ent[i] = lds_entry<T2>(taddr + (uint32_t)(blk * 128));        // [R + immediate]
                    haddr[blk][i] = 2u * taddr + (last ? L.hcL[i] : L.hc4[i]);    // + 256 blk at the point of use
                }
            }
        }
#pragma unroll
        for (int i = 0; i < NSUB; ++i) {
            const bool active = !(last && R == 3) || ((gamma ^ i) < 3);
            if (active) {
                if constexpr (VAR == kVarQ32) {
                    // C4': x = X~_b + Delta~_b r from the fp32 pair, then the integrand's affine variable
                    const double x0 = (double)ent[i].x, dl = (double)ent[i].y;
                    const double r = fma((double)lo[i], 2.3283064365386963e-10, 1.1641532182693481e-10);
                    const double x = fma(dl, r, x0);
                    double sc, sh;
                    if (FID == VEGAS_F_CONST || FID == VEGAS_F_GAUSS) { sc = a.scale[0]; sh = a.shift[0]; }
                    else { const int j = 4 * blk + (gamma ^ i); sc = a.scale[j]; sh = a.shift[j]; }
                    jac[i & (NCH - 1)] *= (T)dl;
                    f.dim((T)((x - sh) * sc), blk, i, ctx);
                } else if constexpr (VAR == kVarU53) {
                    jac[i & (NCH - 1)] *= ent[i].y;
                    f.dim((T)fma((double)ent[i].y, lo53[i], (double)ent[i].x), blk, i, ctx);
                } else {
                    jac[i & (NCH - 1)] *= ent[i].y;
                    f.dim(SP::u(ent[i], lo[i]), blk, i, ctx);
                }
            }
        }
    }
    // events past the end of the launch's range get weight 0 (every built-in f is finite); the weight is ready
    // before f, so only one multiply follows the integrand's tail
    const T jall = chain_prod<NCH, T>(jac);
    if (sizeof(T) == 8) {
        const double wgt = live ? (double)jall * a.post_scale : 0.0;
        const double fv = (double)f.finish(fin0, fin1);
#ifdef VEGAS_USER_INTEGRAND
        if constexpr (FID == VEGAS_F_USER) obs_val = f.observable();     // after finish(): the user's state is complete
#endif
        return fv * wgt;
    }
    (void)jall;
    return (double)f.value(jac, fin0, fin1) * (live ? a.post_scale : 0.0);     // C11: v formed in fp32, then widened
}

// S6 for one event and one section (blocks B0..B1-1), by the warp that holds the section's token: H[j][b_j] += v2 with
// plain loads and stores.  Round i handles sub-step i of every Philox block of the section: within a round the lanes of
// the warp touch pairwise different words (different rows per block; inside a row each lane has its own column), so
// the read-modify-writes of a round are independent and pipeline.  Consecutive rounds can touch the same word from
// different lanes, hence the __syncwarp() (shared memory is processed in order per warp).
template <typename T, int DIM, int B0, int B1, bool PAIR>
__device__ __forceinline__ void rot_hist_update(const uint32_t (&haddr)[(DIM + 3) / 4][4], const uint32_t (&haddrB)[(DIM + 3) / 4][4],
                                                int gammaL, double v2, double v2B) {
    constexpr int NBLK = RotLane<T, DIM>::NBLK, R = RotLane<T, DIM>::R;
    const double v2AB = v2 + v2B;
    (void)v2AB;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        double h[NBLK], hB[NBLK];
        (void)hB;
#pragma unroll
        for (int blk = B0; blk < B1; ++blk) {
            const bool last = (blk == NBLK - 1);
            const int NSUB = last ? ((R == 3) ? 4 : R) : 4;
            const bool active = (i < NSUB) && (!(last && R == 3) || ((gammaL ^ i) < 3));
            if (active) {
                h[blk] = lds_f64(haddr[blk][i] + (uint32_t)(blk * 256));
                if (PAIR) hB[blk] = lds_f64(haddrB[blk][i] + (uint32_t)(blk * 256));
            }
        }
#pragma unroll
        for (int blk = B0; blk < B1; ++blk) {
            const bool last = (blk == NBLK - 1);
            const int NSUB = last ? ((R == 3) ? 4 : R) : 4;
            const bool active = (i < NSUB) && (!(last && R == 3) || ((gammaL ^ i) < 3));
            if (active) {
                if (PAIR) {
                    // two events of this lane in one round: when both fall into the same word the second event's store
                    // goes first and the first event's store, which carries both weights, lands on top of it
                    // (one lane, program order)
                    const bool same = haddr[blk][i] == haddrB[blk][i];
                    sts_f64(haddrB[blk][i] + (uint32_t)(blk * 256), hB[blk] + v2B);
                    sts_f64(haddr[blk][i] + (uint32_t)(blk * 256), h[blk] + (same ? v2AB : v2));
                } else {
                    sts_f64(haddr[blk][i] + (uint32_t)(blk * 256), h[blk] + v2);
                }
            }
        }
        __syncwarp();
    }
}

// the sections of one event's (PAIR: two events') histogram update, each under its own token
template <typename T, int DIM, int SEC, int NSEC, bool MBAR, bool PAIR>
__device__ __forceinline__ void rot_hist_sections(const uint32_t (&haddr)[(DIM + 3) / 4][4], const uint32_t (&haddrB)[(DIM + 3) / 4][4],
                                                  int gammaL, double v2, double v2B, bool ring,
                                                  bool wait, uint32_t my_tok, uint32_t next_tok, uint32_t tok_stride,
                                                  uint32_t parity, bool lane0) {
    if constexpr (SEC < NSEC) {
        constexpr int NBLK = (DIM + 3) / 4;
        if (wait) {
            if (MBAR) token_wait(my_tok + SEC * tok_stride, parity);
            else token_wait_named((int)my_tok);
        }
        rot_hist_update<T, DIM, rot_section_begin(NBLK, NSEC, SEC), rot_section_begin(NBLK, NSEC, SEC + 1), PAIR>(haddr, haddrB, gammaL, v2, v2B);
        if (MBAR) {
            if (ring && lane0) token_pass(next_tok + SEC * tok_stride);     // after the __syncwarp() of the last round
        } else if (ring) {
            token_pass_named((int)next_tok);
        }
        rot_hist_sections<T, DIM, SEC + 1, NSEC, MBAR, PAIR>(haddr, haddrB, gammaL, v2, v2B, ring, wait, my_tok, next_tok, tok_stride, parity, lane0);
    }
}

// The rest of the iteration in the same launch, by CTAs-done tickets in two levels that follow K2's own association:
// the last CTA of slice w (the CTAs w, w+8, w+16, ...) adds that slice's partial rows in K2's fixed order; the last
// slice to finish adds the 8 slice sums in slice order, finalises (S7) and refines (S8).  Which CTA draws the last
// ticket does not matter for the result, and no CTA ever waits for another.  (Not inlined: the event loop's register
// allocation and scheduling stay what they are without it.)
static __device__ __noinline__ void rot_tail(const RotArgs& a, int dim, unsigned char* smem, unsigned int* ticket) {
    const int nb = a.n_bins, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
    const int DIM = dim;
    const int n_parts = (int)gridDim.x, n_tot = 4 + DIM * nb, nent = DIM * nb;
    const int w_me = (int)(blockIdx.x % kReduceSlices);
    const unsigned int in_slice = (unsigned int)((n_parts - w_me + kReduceSlices - 1) / kReduceSlices);
    const unsigned int n_slices = (unsigned int)(n_parts < kReduceSlices ? n_parts : kReduceSlices);
    __threadfence();                                   // this CTA's partial row is visible device-wide ...
    __syncthreads();
    if (threadIdx.x == 0) *ticket = atomicAdd(a.counter + w_me, 1u);      // ... before its ticket is drawn
    __syncthreads();
    if (*ticket != in_slice - 1) return;
    __threadfence();
    double* my_slice = a.slices + (size_t)w_me * nent;
    for (int i = (int)threadIdx.x; i < nent; i += blockDim.x)
        my_slice[i] = reduce_hist_slice(a.partials, n_parts, n_tot, 4 + i, w_me);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) *ticket = atomicAdd(a.counter + kReduceSlices, 1u);
    __syncthreads();
    if (*ticket != n_slices - 1) return;
    __threadfence();
    if (warp == 0) reduce_dd_sum(a.partials, n_parts, n_tot, 0, lane, a.totals);
    if (warp == (nwarps > 1 ? 1 : 0)) reduce_dd_sum(a.partials, n_parts, n_tot, 2, lane, a.totals);
    for (int i = (int)threadIdx.x; i < nent; i += blockDim.x) {
        double t = __ldcg(a.slices + i);
        for (unsigned int w = 1; w < n_slices; ++w) t += __ldcg(a.slices + (size_t)w * nent + i);
        a.totals[4 + i] = t;
    }
    if (threadIdx.x <= kReduceSlices) a.counter[threadIdx.x] = 0u;
    __syncthreads();
    if (threadIdx.x == 0) finalize_result(a.totals, a.tail_n, a.result);
    if (a.tail_alpha >= 0.0) {
        // one warp per dimension, as many at a time as the CTA's shared memory (all of it is free now) has room for
        double* scratch = reinterpret_cast<double*>(smem);
        const int per = (int)refine_scratch_doubles(nb);
        int conc = (int)((size_t)a.tail_smem_doubles / (size_t)per);
        if (conc > nwarps) conc = nwarps;
        if (warp < conc)
            for (int j = warp; j < DIM; j += conc) {
                refine_dimension(const_cast<double*>(a.edges) + (size_t)j * (nb + 1), a.totals + 4 + (size_t)j * nb, nb,
                                 a.tail_alpha, a.status, scratch + (size_t)warp * per, lane, 32, SyncWarp{});
                // refine_dimension ends in a walk of data-dependent length that still reads X[], m[], cum[] of this
                // warp's scratch: every lane must be out of it before the next dimension overwrites them
                __syncwarp();
            }
    }
}

template <int FID, typename T, int DIM, int VAR = 0, bool PAIR = false>
__global__ void __launch_bounds__(rot_max_threads(FID, DIM), 1)
k_iterate_rot(const __grid_constant__ RotArgs a) {
    using T2 = typename RotTableEntry<T, VAR>::type;
    using Lane = RotLane<T, DIM>;
    constexpr int NBLK = Lane::NBLK, GL = Lane::GL;
    constexpr int ENTRY = (int)sizeof(T2);
    extern __shared__ __align__(256) unsigned char smem_rot[];
    const int nb = a.n_bins;
    const int rows = NBLK * nb;
    const int NG = a.n_groups, S = a.ring;
    unsigned char* table = smem_rot;                           // rows x 128 B
    unsigned char* hist = smem_rot + (size_t)rows * 128;       // NG x rows x 256 B
    dd* red = reinterpret_cast<dd*>(hist + (size_t)NG * rows * 256);
    double* obs_sh = reinterpret_cast<double*>(red + 2 * kRotScratchWarps);        // kRotMaxObsBins doubles
    (void)obs_sh;
    constexpr int NSEC = rot_sections(FID, DIM);
    constexpr bool MBAR = rot_mbar_tokens(FID, DIM);
    constexpr bool kPairHold = PAIR;
    const uint32_t tok_base = (uint32_t)__cvta_generic_to_shared(obs_sh + kRotMaxObsBins);   // [NSEC][warp slots] mbarriers
    double* bw_coef = obs_sh + kRotMaxObsBins + kRotMaxSections * kRotScratchWarps;          // BW_POLY beyond 8 dims: [DIM][4]

    // Programmatic dependent launch between the chunk launches of one accumulate call: the next chunk's CTAs may start
    // (prologue, event loop) on SMs this grid has already left; they wait for this grid to complete before they touch
    // the partial rows (griddepcontrol.wait below).  Both instructions are no-ops in an ordinary launch.
    // Where the trigger sits only matters through the code ptxas schedules around it (measured: cfg5 K1 8.72e10 with
    // the trigger here against 8.49e10 after the loop; cfg4 5.15e10 here against 5.24e10 there; cfg3 the same).
    constexpr bool kEarlyTrigger = (FID == VEGAS_F_BW_POLY);
    if (kEarlyTrigger) asm volatile("griddepcontrol.launch_dependents;");
    // ---- prologue: the master grid is staged in shared memory with one coalesced pass (in the histogram region,
    // zeroed afterwards), the table is built from the staged copy, the histograms are zeroed
    {
        double* stage_e = reinterpret_cast<double*>(hist);         // DIM (nb+1) doubles <= one histogram copy
        for (int idx = threadIdx.x; idx < DIM * (nb + 1); idx += blockDim.x) stage_e[idx] = a.edges[idx];
        __syncthreads();
        for (int idx = threadIdx.x; idx < rows * (128 / ENTRY); idx += blockDim.x) {
            const int row = idx / (128 / ENTRY), e = idx - row * (128 / ENTRY);   // entry e of the row
            const int b = row / NBLK, blk = row - b * NBLK;                       // rows are ordered [bin][block]
            const int G = (blk < NBLK - 1) ? 4 : GL;
            const int slot = e / ((128 / ENTRY) / G);
            const int j = 4 * blk + slot;
            T2 ent = T2{};
            if (j < DIM) {
                const double* X = stage_e + j * (nb + 1);
                if constexpr (VAR == kVarU53) ent = RotVarU53::make(X[b], X[b + 1], a.shift[j], a.scale[j]);
                else if constexpr (VAR == kVarQ32) ent = RotVarQ32::make(X[b], X[b + 1]);
                else ent = RotSplit<T, rot_word_map(8 * (int)sizeof(T), DIM)>::make(X[b], X[b + 1], a.shift[j], a.scale[j], b, nb);
            }
            reinterpret_cast<T2*>(table)[idx] = ent;
        }
        __syncthreads();
    }
    for (int idx = threadIdx.x; idx < NG * rows * 32; idx += blockDim.x) reinterpret_cast<double*>(hist)[idx] = 0.0;
    if (FID == VEGAS_F_USER && threadIdx.x < kRotMaxObsBins) obs_sh[threadIdx.x] = 0.0;
    if (FID == VEGAS_F_BW_POLY && DIM > kRotBwMaxDim && threadIdx.x < 4 * DIM)
        bw_coef[threadIdx.x] = a.fpar[5 * (threadIdx.x >> 2) + 1 + (threadIdx.x & 3)];
    if (MBAR && S > 1 && threadIdx.x < NSEC * (blockDim.x >> 5)) {
        token_init(tok_base + 8u * (kRotScratchWarps * (threadIdx.x / (blockDim.x >> 5)) + threadIdx.x % (blockDim.x >> 5)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = warp / S, pos = warp - grp * S;            // histogram copy of this warp, place in its ring
    Lane L;
    L.tbase = (uint32_t)__cvta_generic_to_shared(table);
    {
        const uint32_t hbase = (uint32_t)__cvta_generic_to_shared(hist) + (uint32_t)grp * (uint32_t)rows * 256u;
        const uint32_t toff4 = rot_table_off0<4, ENTRY>(lane), hoff4 = rot_hist_off0<4>(lane);
        const uint32_t toffL = rot_table_off0<GL, ENTRY>(lane), hoffL = rot_hist_off0<GL>(lane);
        constexpr int SHL = (GL == 4) ? 5 : (GL == 2) ? 6 : 7;     // slot -> byte offset shift
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            L.tx4[i] = L.tbase + (toff4 ^ (uint32_t)(i << 5));
            L.txL[i] = L.tbase + (toffL ^ (uint32_t)(i << SHL));
            L.hc4[i] = hbase + (hoff4 ^ (uint32_t)(i << 5)) - 2u * L.tx4[i];
            L.hcL[i] = hbase + (hoffL ^ (uint32_t)(i << SHL)) - 2u * L.txL[i];
        }
    }
    L.gamma4 = rot_gamma<4>(lane);
    L.gammaL = rot_gamma<GL>(lane);
    const T fin0 = (T)a.fin0, fin1 = (T)a.fin1;
    RotCtx<FID, T, NBLK> ctx;
    ctx.init(a, DIM, L.gamma4, L.gammaL);
    if constexpr (FID == VEGAS_F_BW_POLY && DIM > kRotBwMaxDim) ctx.cbase = (uint32_t)__cvta_generic_to_shared(bw_coef);
    constexpr uint32_t tok_stride = 8u * kRotScratchWarps;      // tokens [section][warp slot]: the section is an address immediate
    const int next_warp = grp * S + ((pos + 1 == S) ? 0 : pos + 1);
    uint32_t my_tok = MBAR ? tok_base + 8u * warp : 1u + (uint32_t)warp;              // mbarrier address / barrier id
    uint32_t next_tok = MBAR ? tok_base + 8u * next_warp : 1u + (uint32_t)next_warp;
    // fp64 with mbarrier tokens: kept in two registers; left to itself ptxas rebuilds both addresses from %tid and the
    // shared-memory base at every wait and every hand-off (cfg3 4.16e10 -> 4.33e10 events/s; the named-barrier kernels
    // and the fp32 ones, where ptxas keeps them anyway, lose 1..7 % with the same line: profiles/r02_k1_steps.md)
    if (MBAR && sizeof(T) == 8) {
        asm volatile("" : "+r"(my_tok), "+r"(next_tok));
        asm volatile("" : "+r"(L.tx4[0]), "+r"(L.tx4[1]), "+r"(L.tx4[2]), "+r"(L.tx4[3]));
    }
    const bool ring = S > 1, lane0 = lane == 0;

    // per-thread sums: plain fp64 inside a chunk (a few hundred terms), folded into double-double at the end of every
    // chunk; everything above the thread (warp, CTA, launches, CTAs) is added in double-double too
    // (keeping them in local memory instead frees 8 registers -- 72, enough for 27 warps -- but 27 warps measured
    // 4.20e10 events/s on cfg3 against 4.35e10 with 24, and 21 warps 3.84e10: profiles/r02_k1_steps.md)
    dd a1{0.0, 0.0}, a2{0.0, 0.0};
    // every warp runs the same number of loop iterations (the ring hands the tokens on once per iteration);
    // events past the end of a chunk contribute v = 0
    // The host never lets a launch cross a multiple of 2^32 in the global event index nor exceed 2^32 - 2^20
    // events (vegas_accumulate), so the high counter word of C2 is uniform, the low one is first_lo + q without a
    // carry, and q fits 32 bits even in the padded last pass of the last chunk.
    const uint32_t nthr = gridDim.x * blockDim.x;
    const uint32_t count = (uint32_t)a.count;
    const uint32_t chunk = (a.chunk == 0 || a.chunk > a.count) ? count : (uint32_t)a.chunk;
    const uint32_t e_hi = (uint32_t)(a.first_event >> 32), first_lo = (uint32_t)a.first_event;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    // (waiting unconditionally, with the ring heads' tokens passed once up front, takes the tests of `ring` and `first`
    // out of the loop but measured the same in fp64 and 3 % slower in fp32: profiles/r02_k1_steps.md)
    uint32_t tick = (pos == 0) ? 1u : 0u;      // parity of the token waits: pos 0 skips the wait of its first iteration
    bool first = (pos == 0);
    for (uint32_t c0 = 0, c_end = 0; c0 < count; c0 = c_end) {
        c_end = (count - c0 < chunk) ? count : c0 + chunk;                     // this chunk: events [c0, c_end) of the launch
        const uint32_t n_iter = (c_end - c0 + nthr - 1) / nthr;
        double s1 = 0.0, s2 = 0.0;
        uint32_t q = c0 + tid;
        if (kPairHold && ring) {
            // two events per token hold (rings only): the four dependent read-modify-write rounds of a hold and its
            // hand-off are what a saturated ring is bound by (cfg4: 7 warps per copy); two events share them
            for (uint32_t it = 0; it < n_iter; it += 2, q += 2 * nthr, ++tick) {
                uint32_t haddr[NBLK][4], haddrB[NBLK][4];
                double obs_val = 0.0;
                const double v = rot_event<FID, T, DIM, VAR>(a, L, ctx, first_lo + q, e_hi, q < c_end, fin0, fin1, haddr, obs_val);
                const double vB = rot_event<FID, T, DIM, VAR>(a, L, ctx, first_lo + q + nthr, e_hi, q + nthr < c_end, fin0, fin1, haddrB, obs_val);
                const double v2 = v * v, v2B = vB * vB;
                s1 += v;
                s2 += v2;
                s1 += vB;
                s2 += v2B;
                rot_hist_sections<T, DIM, 0, NSEC, MBAR, true>(haddr, haddrB, L.gammaL, v2, v2B, ring, !first, my_tok, next_tok, tok_stride,
                                                                tick & 1u, lane0);
                first = false;
            }
        } else
        for (uint32_t it = 0; it < n_iter; ++it, q += nthr, ++tick) {
            uint32_t haddr[NBLK][4];
            double obs_val = 0.0;
            const bool live = q < c_end;
            const double v = rot_event<FID, T, DIM, VAR>(a, L, ctx, first_lo + q, e_hi, live, fin0, fin1, haddr, obs_val);
            const double v2 = v * v;
#ifdef VEGAS_USER_INTEGRAND
            if constexpr (FID == VEGAS_F_USER) {
                // observable histogram: one shared-memory add of v per event; v = 0 for padded events
                if (IntegrandU<FID, T, 1>::kObservable && a.n_obs > 0) {
                    const double t = (obs_val - a.obs_lo) * a.obs_inv_width;
                    if (t >= 0.0 && t < (double)a.n_obs && live) atomicAdd(obs_sh + (int)t, v);
                }
            }
#endif
            s1 += v;
            s2 += v2;
            rot_hist_sections<T, DIM, 0, NSEC, MBAR, false>(haddr, haddr, L.gammaL, v2, 0.0, ring, ring && !first, my_tok, next_tok, tok_stride,
                                                            tick & 1u, lane0);
            first = false;
        }
        a1 = dd_add(a1, dd{s1, 0.0});
        a2 = dd_add(a2, dd{s2, 0.0});
    }
    if (!MBAR && ring && pos == 0 && !first) token_wait_named((int)my_tok);   // absorbs the ring's last hand-off
    if (!kEarlyTrigger) asm volatile("griddepcontrol.launch_dependents;");

    // ---- S5: warp shuffle -> CTA -> this CTA's partial (accumulated over the launches of an iteration), all in
    // double-double
    dd t1 = dd_warp_sum(a1), t2 = dd_warp_sum(a2);
    const int nwarps = (blockDim.x + 31) >> 5;
    if (lane == 0) { red[2 * warp] = t1; red[2 * warp + 1] = t2; }
    double* part = a.partials + (size_t)blockIdx.x * (4 + DIM * nb);
    asm volatile("griddepcontrol.wait;" ::: "memory");       // the previous chunk's partial rows are complete
    // this thread's words of the CTA's partial row: loaded now, used after the merge (hides the global latency)
    // (the first 4 words per thread; a shape with more than 4 blockDim.x bins reads the rest in the last pass)
    double own[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int idx = threadIdx.x + k * blockDim.x;
        own[k] = (idx < DIM * nb && !a.overwrite) ? part[4 + idx] : 0.0;
    }
    __syncthreads();
    // warp 0 adds the warps' sums (latency-bound double-double chains) while the other warps merge the histograms
    // (shared-memory-bandwidth-bound); with a single warp it does both
    if (warp == 0) {
        t1 = (lane < nwarps) ? red[2 * lane] : dd{0.0, 0.0};
        t2 = (lane < nwarps) ? red[2 * lane + 1] : dd{0.0, 0.0};
        t1 = dd_warp_sum(t1);
        t2 = dd_warp_sum(t2);
        if (lane == 0) {
            if (!a.overwrite) {
                t1 = dd_add(t1, dd{part[0], part[1]});
                t2 = dd_add(t2, dd{part[2], part[3]});
            }
            part[0] = t1.hi; part[1] = t1.lo; part[2] = t2.hi; part[3] = t2.lo;
        }
    }
    const int mwarps = nwarps > 1 ? nwarps - 1 : 1, mwarp = nwarps > 1 ? warp - 1 : 0;   // merging warps, my rank
    // ---- S6: merge the copies of every (dimension, bin) in fixed order, one pass per CTA.  One warp per
    // histogram row, lane l reads word l of the row (conflict-free; a thread-per-bin loop here put all lanes of
    // a warp on one bank), sums it over the copies, and the words of one dimension slot -- lanes that differ in
    // the half-warp bit and the copy bits -- are added by a fixed xor-shuffle tree.  The row sums are staged in
    // the table's shared memory (dead after the event loop; the barrier above orders it), then added to this
    // CTA's partial row in one coalesced pass.
    double* stage = reinterpret_cast<double*>(table);
    constexpr int LGPL = (GL == 4) ? 2 : (GL == 2) ? 3 : 4;           // log2(copies per slot per half-warp), last block
    const double* hw = reinterpret_cast<const double*>(hist) + lane;
    for (int row0 = mwarp; row0 < rows && mwarp >= 0; row0 += 4 * mwarps) {   // 4 rows in flight per warp
        double h[4] = {0.0, 0.0, 0.0, 0.0};
        for (int g = 0; g < NG; ++g) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int row = row0 + u * mwarps;
                if (row < rows) h[u] += hw[((size_t)g * rows + (size_t)row) * 32];
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            h[u] += __shfl_xor_sync(0xffffffffu, h[u], 16);
            h[u] += __shfl_xor_sync(0xffffffffu, h[u], 1);
            h[u] += __shfl_xor_sync(0xffffffffu, h[u], 2);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int row = row0 + u * mwarps;
            if (row >= rows) continue;                                // warp-uniform
            const int b = row / NBLK, blk = row - b * NBLK;
            const bool last = blk == NBLK - 1;
            const int lgp = last ? LGPL : 2;
            if (lgp >= 3) h[u] += __shfl_xor_sync(0xffffffffu, h[u], 4);
            if (lgp >= 4) h[u] += __shfl_xor_sync(0xffffffffu, h[u], 8);
            const int slot = (lane & 15) >> lgp, c = lane & ((1 << lgp) - 1);
            const int j = 4 * blk + slot;
            if (lane < 16 && c == 0 && j < DIM) stage[j * nb + b] = h[u];
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int idx = threadIdx.x + k * blockDim.x;
        if (idx < DIM * nb) part[4 + idx] = own[k] + stage[idx];
    }
    for (int idx = threadIdx.x + 4 * blockDim.x; idx < DIM * nb; idx += blockDim.x)
        part[4 + idx] = a.overwrite ? stage[idx] : part[4 + idx] + stage[idx];
    // observable bins: one global add per bin per CTA per launch (the order over CTAs is not fixed: 1e-16 effects)
    if (FID == VEGAS_F_USER && a.obs != nullptr && (int)threadIdx.x < a.n_obs) atomicAdd(a.obs + threadIdx.x, obs_sh[threadIdx.x]);

    // ---- the rest of the iteration in the same launch (rot_tail): K2, S7 and S8 by the last CTAs to finish
    if (a.tail) rot_tail(a, DIM, smem_rot, reinterpret_cast<unsigned int*>(red));
}

#ifndef __CUDACC_RTC__
inline size_t rot_shared_bytes(int dim, int n_bins, int n_groups) {
    const size_t rows = (size_t)((dim + 3) / 4) * n_bins;
    return rows * (128 + 256 * (size_t)n_groups) + 2 * sizeof(dd) * kRotScratchWarps +
           sizeof(double) * kRotMaxObsBins + 8 * (size_t)kRotMaxSections * kRotScratchWarps +
           sizeof(double) * 4 * VEGAS_MAX_DIM;
}

// one translation unit per (FID, T, VAR) instantiates DIM = 1..32 (vegas_rot_inst.cu)
template <int FID, typename T, int VAR = 0>
cudaError_t launch_iterate_rot(int dim, const RotArgs& a, int blocks, int threads, size_t shmem, cudaStream_t st);
#endif

}  // namespace vegas
