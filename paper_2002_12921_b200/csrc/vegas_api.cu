// vegas_api.cu -- host driver and C ABI (include/vegas.h) of libvegas_b200.so.
// Chunk loop, launch configuration, workspace carving, parameter derivation, error codes.
// No device allocation, no stream creation, no CPU fallback: every compute entry point launches
// the sm_100a kernels of vegas_kernels.cu or fails with VEGAS_ECUDA.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/vegas.h"
#include "../../include/vegas_instrument.h"
#include "vegas_kernels.h"
#include "vegas_iterate_rot.cuh"
#include "vegas_user.h"

namespace {

constexpr int kMaxBlocks = 1024;      // per-CTA partial slots carved from the workspace
constexpr int kMaxIter = 4096;        // per-iteration result slots (vegas_integrate)
constexpr int kResultStride = 4;      // { I, sigma, status, pad } doubles per iteration
constexpr size_t kAlign = 256;

size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t edges, totals, result, status, hist_up, obs, slices, partials, total;
};

Layout make_layout(int dim, int n_bins) {
    Layout L;
    const size_t nent = (size_t)dim * n_bins, ntot = 4 + nent;
    size_t off = 0;
    L.edges = off;    off += align_up(sizeof(double) * dim * (n_bins + 1));
    L.totals = off;   off += align_up(sizeof(double) * ntot);
    L.result = off;   off += align_up(sizeof(double) * kResultStride * kMaxIter);
    L.status = off;   off += align_up(sizeof(int) * 32);    // [0] refinement status, [8..16] CTAs-done tickets
    L.hist_up = off;  off += align_up(sizeof(double) * nent);
    L.obs = off;      off += align_up(sizeof(double) * vegas::kRotMaxObsBins);
    L.slices = off;   off += align_up(sizeof(double) * nent * vegas::kReduceSlices);
    L.partials = off; off += align_up(sizeof(double) * ntot * kMaxBlocks);
    L.total = off;
    return L;
}

bool valid_shape(int dim, int n_bins) {
    return dim >= 1 && dim <= VEGAS_MAX_DIM && n_bins >= 2 && n_bins <= VEGAS_MAX_BINS;
}

int expected_n_params(int fid, int dim) {
    switch (fid) {
    case VEGAS_F_CONST: return 0;
    case VEGAS_F_GAUSS: return 1;
    case VEGAS_F_GENZ_PRODUCT_PEAK: return 2 * dim;
    case VEGAS_F_GENZ_DISCONTINUOUS: return 2 * dim;
    case VEGAS_F_BW_POLY: return dim >= 2 ? 4 + 5 * (dim - 1) : -1;
    default: return -1;
    }
}

}  // namespace

struct vegas_grid {
    int dim = 0, n_bins = 0, device = 0, sm_count = 0;
    size_t smem_optin = 0, smem_total_sm = 0;
    unsigned char* ws = nullptr;
    Layout L{};
    double* d_edges = nullptr;
    double* d_totals = nullptr;
    double* d_result = nullptr;
    int* d_status = nullptr;
    double* d_hist_up = nullptr;
    double* d_partials = nullptr;
    unsigned int* d_counter = nullptr;           // CTAs-done tickets of the one-launch iteration
    double* d_slices = nullptr;                  // its slice sums (K2's association)
    double* d_obs = nullptr;                     // observable histogram of a user integrand: sums of v per bin
    int n_obs = 0;
    double obs_lo = 0.0, obs_hi = 1.0;
    bool params_set[6] = {true, false, false, false, false, false};
    double derived[6][VEGAS_MAX_PARAMS] = {};
    double user[6][VEGAS_MAX_PARAMS] = {};       // the caller's arrays as given to vegas_set_params
    vegas::UserKernel ukernel;                   // VEGAS_F_USER: the run-time compiled fused kernel
    int cfg_blocks = 0, cfg_threads = 0, cfg_ct = 0, cfg_ch = 0;
    double* h_cb = nullptr;         // page-locked HOST staging of the host-callback path (x and f of two batches)
    size_t h_cb_doubles = 0;
    cudaEvent_t cb_ev[4] = {nullptr, nullptr, nullptr, nullptr};     // its "x arrived" / "f consumed" events, per slot
    double* h_pinned = nullptr;     // page-locked HOST staging for the per-iteration results of vegas_integrate (a copy to
                                    // pageable memory costs ~10 us more per call); host memory, owned by the library
    int variant = 0;                // VEGAS_VARIANT_*: the sampling map of the iterate calls (vegas_set_variant)
    int active_blocks = 0;          // CTAs whose partial slots the current iteration uses
    bool profiling = false;
    std::vector<cudaEvent_t> events;   // pairs (start, stop)
    size_t events_used = 0;
    double kernel_ms_acc = 0.0;
    uint64_t iterate_launches = 0, launches = 0;
    char cuda_err[256] = "";
};

namespace {

int cuda_fail(vegas_grid* g, cudaError_t e, const char* what) {
    if (g) snprintf(g->cuda_err, sizeof(g->cuda_err), "%s: %s", what, cudaGetErrorString(e));
    return VEGAS_ECUDA;
}

#define CUDA_TRY(g, call)                                        \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return cuda_fail(g, e__, #call); \
    } while (0)

struct LaunchShape {
    int blocks, threads, ct, ch;
    size_t shmem;
};

// Predicted shared-pipe cost (SM clocks per warp-wide access) of the table gather and of the
// histogram CAS update as a function of the copy count, from the step-0 microbenchmarks on a
// B200 (profiles/r01_s7_ubench_pipes.md).  Only used to rank (ct, ch) pairs that fit.
double table_cost(int precision, int ct) {
    static const double c64[] = {9.5, 9.4, 7.9, 6.5, 6.5, 6.5};     // ct = 1,2,4,8,(16,32)
    static const double c32[] = {6.0, 5.6, 5.0, 4.2, 3.4, 3.4};
    int l = 0;
    while ((1 << l) < ct) ++l;
    return precision == VEGAS_FP64 ? c64[l] : c32[l];
}
double hist_cost(int ch) {
    static const double c[] = {26.0, 23.5, 20.0, 15.5, 9.7, 9.0};   // ch = 1,2,4,8,16,32
    int l = 0;
    while ((1 << l) < ch) ++l;
    return c[l];
}

int resolve_launch(const vegas_grid* g, int precision, LaunchShape* out) {
    LaunchShape s;
    s.blocks = g->cfg_blocks > 0 ? g->cfg_blocks : g->sm_count;
    s.threads = g->cfg_threads > 0 ? g->cfg_threads : vegas::kIterMaxThreads;
    if (s.blocks > kMaxBlocks || s.threads > 1024 || s.threads % 32) return VEGAS_EINVAL;
    if (s.threads > vegas::kIterMaxThreads) s.threads = vegas::kIterMaxThreads;   // the generic kernel's launch bound
    const int max_ct = precision == VEGAS_FP64 ? 8 : 16;
    double best = 1e300;
    s.ct = s.ch = 0;
    for (int ch = 1; ch <= 32; ch *= 2) {
        if (g->cfg_ch > 0 && ch != g->cfg_ch) continue;
        if (g->cfg_ch == 0 && ch > 16) continue;
        for (int ct = 1; ct <= 32; ct *= 2) {
            if (g->cfg_ct > 0 && ct != g->cfg_ct) continue;
            if (g->cfg_ct == 0 && ct > max_ct) continue;
            const size_t sh = vegas::iterate_shared_bytes(g->dim, g->n_bins, precision, ct, ch);
            if (sh > g->smem_optin) continue;
            const double cost = table_cost(precision, ct) + hist_cost(ch) + 1e-9 * (double)sh;
            if (cost < best) { best = cost; s.ct = ct; s.ch = ch; s.shmem = sh; }
        }
    }
    if (s.ct == 0) return VEGAS_EINVAL;
    *out = s;
    return VEGAS_OK;
}

int ilog2(int v) {
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

bool use_rot_path(const vegas_grid* g, int fid, int precision);
// the variants of the sampling map exist as fp64 fast-path kernels of the built-in integrands
bool variant_available(const vegas_grid* g, int fid, int precision) {
    return precision == VEGAS_FP64 && fid != VEGAS_F_USER && fid != VEGAS_F_GENZ_DISCONTINUOUS && use_rot_path(g, fid, precision);
}

bool check_call(const vegas_grid* g, int fid, int precision) {
    if (!g) return false;
    if (fid < 0 || fid > VEGAS_F_GENZ_DISCONTINUOUS || !g->params_set[fid]) return false;
    if (fid == VEGAS_F_USER) return g->ukernel.kernel != nullptr && (precision == VEGAS_FP64 || precision == VEGAS_FP32) && g->variant == 0;
    if (expected_n_params(fid, g->dim) < 0) return false;
    if (g->variant != 0 && !variant_available(g, fid, precision)) return false;
    if (fid == VEGAS_F_GENZ_DISCONTINUOUS) return precision == VEGAS_FP64;      // the cuts are decided in fp64 (vegas.h)
    return precision == VEGAS_FP64 || precision == VEGAS_FP32;
}

double jac_scale_for(const vegas_grid* g, int precision) {
    if (precision != VEGAS_FP64) return 1.0;
    double s = 1.0;
    for (int j = 0; j < g->dim; ++j) s *= (double)g->n_bins;
    return s;
}

// The fast path (vegas_iterate_rot.cuh) serves integrands that are functions of per-dimension affine
// variables; it is taken unless the caller pinned the copy counts of the generic kernel with
// vegas_set_launch (which is also how the tests keep the generic kernel covered).
bool use_rot_path(const vegas_grid* g, int fid, int precision) {
    if (fid == VEGAS_F_USER) return true;          // a user integrand exists only as a fast-path kernel
    if (g->cfg_ct > 0 || g->cfg_ch > 0) return false;
    (void)precision;
    const bool kind = fid == VEGAS_F_CONST || fid == VEGAS_F_GAUSS || fid == VEGAS_F_GENZ_PRODUCT_PEAK ||
                      fid == VEGAS_F_BW_POLY || fid == VEGAS_F_GENZ_DISCONTINUOUS;
    if (!kind) return false;
    return vegas::rot_shared_bytes(g->dim, g->n_bins, 1) <= g->smem_optin;
}

// shift_j, scale_j, post_scale, fin0 of the affine pre-composition (see vegas_iterate_rot.cuh)
void rot_constants(const vegas_grid* g, int fid, int precision, double* shift, double* scale, double* post_scale,
                   double* fin0, double* fin1, double* jac_init, double* fpar, bool word_map, int variant = 0) {
    const int dim = g->dim;
    const double nb = (double)g->n_bins;
    *post_scale = 1.0;
    *fin0 = 0.0;
    *fin1 = 0.0;
    for (int j = 0; j < VEGAS_MAX_DIM; ++j) { shift[j] = 0.0; scale[j] = nb; }
    if (fid == VEGAS_F_GAUSS) {
        const double a = g->user[fid][0];
        for (int j = 0; j < dim; ++j) shift[j] = 0.5;
        *fin0 = 1.0 / ((nb * a) * (nb * a));
        *post_scale = g->derived[fid][0];                       // (a sqrt(pi))^-d; prod B_j is the Jacobian
        if (precision == VEGAS_FP32) {
            // fp32 (C11): ln N goes into the exponent (IntegrandU<GAUSS>::finish); what its rounding to fp32 leaves
            // of N, a factor 1 +- 2e-6, stays here and is applied after the widening
            const double ln_n = -(double)dim * std::log(a * std::sqrt(3.14159265358979323846));
            const float ln_n32 = (float)ln_n;
            *fin1 = (double)ln_n32;
            *post_scale = std::exp(ln_n - (double)ln_n32);
        }
    } else if (fid == VEGAS_F_GENZ_PRODUCT_PEAK) {
        double ps = 1.0;
        for (int j = 0; j < dim; ++j) {
            const double c = g->user[fid][j];
            shift[j] = g->user[fid][dim + j];
            scale[j] = c;
            ps *= c * nb;                                        // f J = prod(c_j nb) prod B_j / prod(1+u_j^2)
        }
        *post_scale = ps;
        if (precision == VEGAS_FP32) {
            // fp32 (C11): n_bins^d is shared out over the four chains (IntegrandU<GENZ>::value), prod c_j stays here
            const float q32 = (float)std::pow(nb, 0.25 * dim);
            double pc = 1.0;
            for (int j = 0; j < dim; ++j) pc *= g->user[fid][j];
            *fin1 = (double)q32;
            *post_scale = pc * std::exp((double)dim * std::log(nb) - 4.0 * std::log((double)q32));
        }
    } else if (fid == VEGAS_F_GENZ_DISCONTINUOUS) {
        double ps = 1.0, k = 0.0;                                // u_j = c_j (x_j - a_j): J = prod (nb / c_j) B_j 2^32
        for (int j = 0; j < dim; ++j) {
            const double c = g->user[fid][j], a = g->user[fid][dim + j];
            shift[j] = a;
            scale[j] = c;
            ps *= nb / c;
            k += c * a;
        }
        *post_scale = ps;
        *fin1 = k;                                               // exp(sum c_j x_j) = exp(sum u_j + sum c_j a_j)
    } else if (fid == VEGAS_F_USER) {
        double ps = 1.0;                                         // u_j = x_j; J = prod nb Delta_j = nb^d prod B_j 2^32
        for (int j = 0; j < dim; ++j) { scale[j] = 1.0; ps *= nb; }
        *post_scale = ps;
        if (precision == VEGAS_FP32) {
            // fp32 (C11): n_bins^d is shared out over the four chains (IntegrandU<USER>::value)
            const float q32 = (float)std::pow(nb, 0.25 * dim);
            *fin1 = (double)q32;
            *post_scale = std::exp((double)dim * std::log(nb) - 4.0 * std::log((double)q32));
        }
        for (int k = 0; k < vegas::kRotParams; ++k) fpar[k] = g->user[fid][k];
    } else if (fid == VEGAS_F_BW_POLY) {
        // u_0 = (s - M^2)/(M Gamma) with s = s_min + x_0 ds (C5): the Breit-Wigner is 1/(1 + u_0^2); u_j = x_j, j >= 1
        const double* d = g->derived[fid];                       // s_min, ds, M^2, M^2 Gamma^2, a[i][k]
        const double mg = std::sqrt(d[3]);
        shift[0] = (d[2] - d[0]) / d[1];
        scale[0] = d[1] / mg;
        double ps = nb / scale[0];
        for (int j = 1; j < dim; ++j) { scale[j] = 1.0; ps *= nb; }
        *post_scale = ps;                                        // J = prod nb Delta_j = prod (nb/scale_j) B_j 2^32
        if (precision == VEGAS_FP32) {
            // fp32 (C11): n_bins^d is shared out over the four chains (IntegrandU<BW_POLY>::value)
            const float q32 = (float)std::pow(nb, 0.25 * dim);
            *fin1 = (double)q32;
            *post_scale = std::exp((double)dim * std::log(nb) - 4.0 * std::log((double)q32)) / scale[0];
        }
        for (int k = 0; k < 5; ++k) fpar[k] = 0.0;               // row 0: the Breit-Wigner dimension has no polynomial
        for (int j = 1; j < dim; ++j)
            for (int k = 0; k < 5; ++k) fpar[5 * j + k] = d[4 + 5 * (j - 1) + k];
    }
    // fp64 table entries carry 2^-32 per dimension (RotEntry<double>): start the running Jacobian product at
    // 2^(32 floor(d/2)) and give the rest back in post_scale -- exact powers of two, the product stays in range
    *jac_init = 1.0;
    if (precision == VEGAS_FP64 && variant == VEGAS_VARIANT_Q32) {
        // C4': the table holds (X~_b, Delta~_b) themselves; the running product is prod Delta~_b and
        // J = n_bins^d prod Delta~_b, so the scale_j and n_bins that the other tables carry in B come back here
        for (int j = 0; j < dim; ++j) *post_scale *= scale[j];
    } else if (precision == VEGAS_FP64) {
        const int h = dim / 2, bits = vegas::rot_jac_bits(64, variant);      // 2^-32 per dimension, 2^-53 for C3'
        *jac_init = std::ldexp(1.0, bits * h);
        *post_scale *= std::ldexp(1.0, bits * (dim - h));
        // the fast path's fp64 table entries are affine in the whole Philox word (RotEntry<double>::make_w): their
        // slope, the Jacobian factor, carries one more n_bins per dimension
        if (word_map && variant == 0)
            for (int j = 0; j < dim; ++j) *post_scale /= nb;
    }
}

struct RotShape {
    int blocks, threads, n_groups, ring;
    size_t shmem;
};

// what the last CTA of a one-launch iteration does after the event loop (vegas_iterate_rot.cuh: RotArgs::tail)
struct Tail {
    double n_events, alpha;     // alpha < 0: no refinement
    double* d_result;           // device, { I, sigma, status }
};
int accumulate_impl(vegas_grid* g, uint64_t first_event, uint64_t count, uint64_t chunk_events, uint64_t seed,
                    uint32_t iteration, int fid, int precision, void* cuda_stream, const Tail* tail);

// One CTA per SM.  n_groups = histogram copies in the CTA (as many as fit next to the table, a divisor of the warp
// count W), ring = W / n_groups warps share a copy (1 = no token passing).  W is the caller's choice (vegas_set_launch),
// else: with mbarrier tokens (24-warp kernels) the warp count among the four largest that gives the most copies; with
// named-barrier tokens (16-warp kernels) 16 when every warp can own a copy, otherwise the largest of 15..12 that keeps
// more than half of the copies that fit (measured on B200, profiles/r01_s13_fast_path.md).
static int rot_divisor(int W, int fit) {
    int ng = fit < W ? fit : W;
    while (W % ng) --ng;
    return ng;
}
RotShape rot_shape(const vegas_grid* g, int fid) {
    RotShape s;
    const size_t one = vegas::rot_shared_bytes(g->dim, g->n_bins, 1), base = vegas::rot_shared_bytes(g->dim, g->n_bins, 0);
    int fit = (int)((g->smem_optin - base) / (one - base));
    if (fit < 1) fit = 1;
    const int wmax = vegas::rot_max_warps(fid, g->dim);
    const bool mbar = vegas::rot_mbar_tokens(fid, g->dim);
    int W = wmax;
    if (g->cfg_threads > 0) {
        W = (g->cfg_threads + 31) / 32;
        if (W > wmax) W = wmax;                        // the kernel's launch bound (a user kernel is built for 12 warps)
        if (!mbar && fit < W && W > vegas::kRotMaxNamedRingWarps) W = vegas::kRotMaxNamedRingWarps;
    } else if (mbar) {
        int best = 0;
        for (int w = wmax; w > wmax - 4 && w >= 1; --w) {
            const int ng = rot_divisor(w, fit);
            if (ng > best) { best = ng; W = w; }
        }
    } else if (fit < wmax) {
        W = vegas::kRotNamedDefaultWarps < wmax ? vegas::kRotNamedDefaultWarps : wmax;
        const int top = wmax - 1 < vegas::kRotMaxNamedRingWarps ? wmax - 1 : vegas::kRotMaxNamedRingWarps;
        for (int w = top; w > W; --w)
            if (2 * rot_divisor(w, fit) > fit) { W = w; break; }
    }
    const int ng = rot_divisor(W, fit);
    s.n_groups = ng;
    s.ring = W / ng;
    s.threads = 32 * W;
    s.shmem = vegas::rot_shared_bytes(g->dim, g->n_bins, ng);
    s.blocks = g->cfg_blocks > 0 ? g->cfg_blocks : g->sm_count;
    return s;
}

cudaError_t launch_rot(vegas_grid* g, int fid, int precision, int dim, const vegas::RotArgs& a, const RotShape& s,
                       cudaStream_t st) {
    if (fid == VEGAS_F_USER) return vegas::user_launch(&g->ukernel, precision == VEGAS_FP32, a, s.blocks, s.threads, s.shmem, st);
    if (precision == VEGAS_FP64 && g->variant != 0) {
#define VEGAS_VAR_CASE(F)                                                                                              \
    case F:                                                                                                            \
        return g->variant == VEGAS_VARIANT_U53                                                                         \
                   ? vegas::launch_iterate_rot<F, double, vegas::kVarU53>(dim, a, s.blocks, s.threads, s.shmem, st)    \
                   : vegas::launch_iterate_rot<F, double, vegas::kVarQ32>(dim, a, s.blocks, s.threads, s.shmem, st);
        switch (fid) {
            VEGAS_VAR_CASE(VEGAS_F_CONST)
            VEGAS_VAR_CASE(VEGAS_F_GAUSS)
            VEGAS_VAR_CASE(VEGAS_F_GENZ_PRODUCT_PEAK)
            VEGAS_VAR_CASE(VEGAS_F_BW_POLY)
        }
#undef VEGAS_VAR_CASE
        return cudaErrorInvalidValue;
    }
    if (precision == VEGAS_FP64) {
        switch (fid) {
        case VEGAS_F_CONST: return vegas::launch_iterate_rot<VEGAS_F_CONST, double>(dim, a, s.blocks, s.threads, s.shmem, st);
        case VEGAS_F_GAUSS: return vegas::launch_iterate_rot<VEGAS_F_GAUSS, double>(dim, a, s.blocks, s.threads, s.shmem, st);
        case VEGAS_F_GENZ_PRODUCT_PEAK:
            return vegas::launch_iterate_rot<VEGAS_F_GENZ_PRODUCT_PEAK, double>(dim, a, s.blocks, s.threads, s.shmem, st);
        case VEGAS_F_BW_POLY:
            return vegas::launch_iterate_rot<VEGAS_F_BW_POLY, double>(dim, a, s.blocks, s.threads, s.shmem, st);
        case VEGAS_F_GENZ_DISCONTINUOUS:
            return vegas::launch_iterate_rot<VEGAS_F_GENZ_DISCONTINUOUS, double>(dim, a, s.blocks, s.threads, s.shmem, st);
        }
    } else {
        switch (fid) {
        case VEGAS_F_CONST: return vegas::launch_iterate_rot<VEGAS_F_CONST, float>(dim, a, s.blocks, s.threads, s.shmem, st);
        case VEGAS_F_GAUSS: return vegas::launch_iterate_rot<VEGAS_F_GAUSS, float>(dim, a, s.blocks, s.threads, s.shmem, st);
        case VEGAS_F_GENZ_PRODUCT_PEAK:
            return vegas::launch_iterate_rot<VEGAS_F_GENZ_PRODUCT_PEAK, float>(dim, a, s.blocks, s.threads, s.shmem, st);
        case VEGAS_F_BW_POLY:
            return vegas::launch_iterate_rot<VEGAS_F_BW_POLY, float>(dim, a, s.blocks, s.threads, s.shmem, st);
        }
    }
    return cudaErrorInvalidValue;
}

int fetch_result(vegas_grid* g, cudaStream_t st, double* I, double* sigma, double* hist_host);

int finish_iteration(vegas_grid* g, uint64_t n_total, cudaStream_t st, double* I, double* sigma, double* hist_host) {
    CUDA_TRY(g, vegas::launch_finalize(g->d_totals, (double)n_total, g->d_result, st));
    g->launches++;
    return fetch_result(g, st, I, sigma, hist_host);
}

// D2H of { I, sigma, status } (and the histogram totals), one synchronisation
int fetch_result(vegas_grid* g, cudaStream_t st, double* I, double* sigma, double* hist_host) {
    const size_t nent = (size_t)g->dim * g->n_bins;
    double res[3] = {0, 0, 0};
    CUDA_TRY(g, cudaMemcpyAsync(res, g->d_result, sizeof(res), cudaMemcpyDeviceToHost, st));
    if (hist_host)
        CUDA_TRY(g, cudaMemcpyAsync(hist_host, g->d_totals + 4, sizeof(double) * nent, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    if (I) *I = res[0];
    if (sigma) *sigma = res[1];
    return res[2] == 0.0 ? VEGAS_OK : VEGAS_ENUMERIC;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

size_t vegas_workspace_bytes(int dim, int n_bins) {
    if (!valid_shape(dim, n_bins)) return 0;
    return make_layout(dim, n_bins).total;
}

int vegas_create(int dim, int n_bins, void* dev_workspace, size_t bytes, vegas_grid** out) {
    if (!out) return VEGAS_EINVAL;
    *out = nullptr;
    if (!valid_shape(dim, n_bins) || !dev_workspace) return VEGAS_EINVAL;
    if (((uintptr_t)dev_workspace) % kAlign) return VEGAS_EINVAL;
    const Layout L = make_layout(dim, n_bins);
    if (bytes < L.total) return VEGAS_EINVAL;
    vegas_grid* g = new (std::nothrow) vegas_grid();
    if (!g) return VEGAS_EINVAL;
    cudaError_t e = cudaGetDevice(&g->device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, g->device);
    if (e != cudaSuccess) { delete g; return VEGAS_ECUDA; }
    g->dim = dim;
    g->n_bins = n_bins;
    g->sm_count = prop.multiProcessorCount;
    g->smem_optin = prop.sharedMemPerBlockOptin;
    g->smem_total_sm = prop.sharedMemPerMultiprocessor;
    g->ws = (unsigned char*)dev_workspace;
    g->L = L;
    g->d_edges = (double*)(g->ws + L.edges);
    g->d_totals = (double*)(g->ws + L.totals);
    g->d_result = (double*)(g->ws + L.result);
    g->d_status = (int*)(g->ws + L.status);
    g->d_counter = (unsigned int*)(g->d_status + 8);
    g->d_slices = (double*)(g->ws + L.slices);
    g->d_hist_up = (double*)(g->ws + L.hist_up);
    g->d_partials = (double*)(g->ws + L.partials);
    g->d_obs = (double*)(g->ws + L.obs);
    std::vector<double> edges((size_t)dim * (n_bins + 1));
    for (int j = 0; j < dim; ++j)
        for (int i = 0; i <= n_bins; ++i) edges[(size_t)j * (n_bins + 1) + i] = (double)i / (double)n_bins;
    e = cudaMemcpy(g->d_edges, edges.data(), sizeof(double) * edges.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(g->d_totals, 0, L.slices - L.totals);      // totals .. observable sums
    if (e != cudaSuccess) { delete g; return VEGAS_ECUDA; }
    *out = g;
    return VEGAS_OK;
}

int vegas_destroy(vegas_grid* g) {
    if (!g) return VEGAS_EINVAL;
    for (cudaEvent_t ev : g->events) cudaEventDestroy(ev);
    if (g->h_pinned) cudaFreeHost(g->h_pinned);
    if (g->h_cb) cudaFreeHost(g->h_cb);
    for (cudaEvent_t ev : g->cb_ev)
        if (ev) cudaEventDestroy(ev);
    vegas::user_unload(&g->ukernel);
    delete g;
    return VEGAS_OK;
}

int vegas_set_params(vegas_grid* g, int fid, const double* p, int n_params) {
    // everything is validated into temporaries: a rejected call leaves the grid's parameters as they were
    if (g && fid == VEGAS_F_USER) {
        if (n_params < 0 || n_params > VEGAS_USER_MAX_PARAMS || (n_params > 0 && !p)) return VEGAS_EINVAL;
        for (int i = 0; i < n_params; ++i)
            if (!std::isfinite(p[i])) return VEGAS_EINVAL;
        std::memset(g->user[fid], 0, sizeof(g->user[fid]));
        for (int i = 0; i < n_params; ++i) g->user[fid][i] = p[i];
        g->params_set[fid] = true;
        return VEGAS_OK;
    }
    if (!g || fid < 0 || (fid > 3 && fid != VEGAS_F_GENZ_DISCONTINUOUS)) return VEGAS_EINVAL;
    const int want = expected_n_params(fid, g->dim);
    if (want < 0 || n_params != want || want > VEGAS_MAX_PARAMS || (want > 0 && !p)) return VEGAS_EINVAL;
    for (int i = 0; i < want; ++i)
        if (!std::isfinite(p[i])) return VEGAS_EINVAL;
    double d[VEGAS_MAX_PARAMS] = {};
    const int dim = g->dim;
    switch (fid) {
    case VEGAS_F_CONST: break;
    case VEGAS_F_GAUSS: {
        const double a = p[0];
        if (!(a > 0.0)) return VEGAS_EINVAL;
        d[0] = std::pow(a * std::sqrt(3.14159265358979323846), -(double)dim);
        d[1] = 1.0 / (a * a);
        break;
    }
    case VEGAS_F_GENZ_PRODUCT_PEAK:
        for (int j = 0; j < dim; ++j) {
            if (p[j] == 0.0) return VEGAS_EINVAL;
            d[2 * j] = 1.0 / (p[j] * p[j]);
            d[2 * j + 1] = p[dim + j];
        }
        break;
    case VEGAS_F_GENZ_DISCONTINUOUS:
        for (int j = 0; j < dim; ++j)
            if (!(p[j] > 0.0)) return VEGAS_EINVAL;                      // c_j > 0: the cut is u_j <= 0 on the fast path
        break;
    case VEGAS_F_BW_POLY: {
        const double M = p[0], G = p[1], m_min = p[2], m_max = p[3];
        d[0] = m_min * m_min;
        d[1] = m_max * m_max - m_min * m_min;
        d[2] = M * M;
        d[3] = M * M * G * G;
        if (!(d[3] > 0.0) || !(d[1] > 0.0)) return VEGAS_EINVAL;       // M Gamma != 0, m_max^2 > m_min^2
        for (int i = 0; i < 5 * (dim - 1); ++i) d[4 + i] = p[4 + i];
        break;
    }
    }
    std::memcpy(g->derived[fid], d, sizeof(d));
    std::memset(g->user[fid], 0, sizeof(g->user[fid]));
    for (int i = 0; i < want; ++i) g->user[fid][i] = p[i];
    g->params_set[fid] = true;
    return VEGAS_OK;
}

int vegas_set_user_integrand(vegas_grid* g, const char* cuda_source, const double* params_host, int n_params,
                             char* log, size_t log_bytes) {
    if (log && log_bytes) log[0] = '\0';
    if (!g || !cuda_source) return VEGAS_EINVAL;
    if (vegas::rot_shared_bytes(g->dim, g->n_bins, 1) > g->smem_optin) return VEGAS_EINVAL;
    if (n_params < 0 || n_params > VEGAS_USER_MAX_PARAMS || (n_params > 0 && !params_host)) return VEGAS_EINVAL;
    for (int i = 0; i < n_params; ++i)
        if (!std::isfinite(params_host[i])) return VEGAS_EINVAL;
    CUDA_TRY(g, cudaSetDevice(g->device));
    std::string clog, err;
    vegas::UserKernel fresh;                         // the old kernel and its parameters stay until this one is ready
    const int rc = vegas::user_compile(cuda_source, g->dim, &clog, &fresh, &err);
    if (log && log_bytes) {
        const std::string& msg = clog.empty() ? err : clog;
        snprintf(log, log_bytes, "%s", msg.c_str());
    }
    if (rc != 0) {
        snprintf(g->cuda_err, sizeof(g->cuda_err), "%s", err.c_str());
        return rc == -1 ? VEGAS_EINVAL : VEGAS_ECUDA;
    }
    vegas::user_unload(&g->ukernel);
    g->ukernel = fresh;
    return vegas_set_params(g, VEGAS_F_USER, params_host, n_params);
}

int vegas_set_observable(vegas_grid* g, double lo, double hi, int n_obs_bins) {
    if (!g || n_obs_bins < 0 || n_obs_bins > vegas::kRotMaxObsBins) return VEGAS_EINVAL;
    if (n_obs_bins > 0 && (!(hi > lo) || !std::isfinite(lo) || !std::isfinite(hi))) return VEGAS_EINVAL;
    g->n_obs = n_obs_bins;
    g->obs_lo = lo;
    g->obs_hi = hi;
    return VEGAS_OK;
}

int vegas_get_observable_hist(vegas_grid* g, double* obs_hist_host, void* cuda_stream) {
    if (!g || !obs_hist_host || g->n_obs <= 0) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    CUDA_TRY(g, cudaMemcpyAsync(obs_hist_host, g->d_obs, sizeof(double) * g->n_obs, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    return VEGAS_OK;
}

int vegas_set_edges(vegas_grid* g, const double* edges_host, void* cuda_stream) {
    if (!g || !edges_host) return VEGAS_EINVAL;
    const int nb = g->n_bins;
    for (int j = 0; j < g->dim; ++j) {
        const double* X = edges_host + (size_t)j * (nb + 1);
        if (X[0] != 0.0 || X[nb] != 1.0) return VEGAS_EINVAL;
        for (int i = 0; i < nb; ++i)
            if (!(X[i + 1] > X[i])) return VEGAS_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    CUDA_TRY(g, cudaMemcpyAsync(g->d_edges, edges_host, sizeof(double) * g->dim * (nb + 1), cudaMemcpyHostToDevice, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    return VEGAS_OK;
}

int vegas_get_edges(vegas_grid* g, double* edges_host, void* cuda_stream) {
    if (!g || !edges_host) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    CUDA_TRY(g, cudaMemcpyAsync(edges_host, g->d_edges, sizeof(double) * g->dim * (g->n_bins + 1), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    return VEGAS_OK;
}

int vegas_get_hist(vegas_grid* g, double* hist_host, void* cuda_stream) {
    if (!g || !hist_host) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    CUDA_TRY(g, cudaMemcpyAsync(hist_host, g->d_totals + 4, sizeof(double) * g->dim * g->n_bins, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    return VEGAS_OK;
}

int vegas_begin_iteration(vegas_grid* g, void* cuda_stream) {
    if (!g) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    LaunchShape s;
    if (resolve_launch(g, VEGAS_FP64, &s)) return VEGAS_EINVAL;
    // either kernel path may serve the accumulate calls of this iteration: reserve slots for the wider one
    int blocks = s.blocks;
    if (use_rot_path(g, VEGAS_F_CONST, VEGAS_FP64)) {
        const RotShape r = rot_shape(g, VEGAS_F_CONST);
        if (r.blocks > blocks) blocks = r.blocks;
    }
    if (blocks > kMaxBlocks) return VEGAS_EINVAL;
    g->active_blocks = blocks;
    const size_t ntot = 4 + (size_t)g->dim * g->n_bins;
    CUDA_TRY(g, cudaMemsetAsync(g->d_partials, 0, sizeof(double) * ntot * blocks, st));
    CUDA_TRY(g, cudaMemsetAsync(g->d_obs, 0, sizeof(double) * vegas::kRotMaxObsBins, st));
    return VEGAS_OK;
}

int vegas_accumulate(vegas_grid* g, uint64_t first_event, uint64_t count, uint64_t chunk_events, uint64_t seed,
                     uint32_t iteration, int fid, int precision, void* cuda_stream) {
    return accumulate_impl(g, first_event, count, chunk_events, seed, iteration, fid, precision, cuda_stream, nullptr);
}

}  // extern "C"
#pragma GCC visibility pop

namespace {

// Can a whole iteration of n events from event 0 run as one fast-path launch (reduce, finalize and refine fused into it)?
bool one_launch_iteration(const vegas_grid* g, uint64_t n_events, int fid, int precision) {
    return use_rot_path(g, fid, precision) && n_events <= 0xFFF00000ull;
}

// One iteration in the stream, not synchronised: totals, result slot (and the refined grid if alpha >= 0) on the device.
int enqueue_iteration(vegas_grid* g, uint64_t n_events, uint64_t chunk_events, uint64_t seed, uint32_t iteration, int fid,
                      int precision, cudaStream_t st, double alpha, double* d_result) {
    if (one_launch_iteration(g, n_events, fid, precision)) {
        const RotShape rs = rot_shape(g, fid);
        if (rs.blocks > kMaxBlocks) return VEGAS_EINVAL;
        g->active_blocks = rs.blocks;
        if (g->n_obs > 0) CUDA_TRY(g, cudaMemsetAsync(g->d_obs, 0, sizeof(double) * vegas::kRotMaxObsBins, st));
        const Tail tail{(double)n_events, alpha, d_result};
        return accumulate_impl(g, 0, n_events, chunk_events, seed, iteration, fid, precision, (void*)st, &tail);
    }
    int rc = vegas_begin_iteration(g, (void*)st);
    if (rc) return rc;
    rc = accumulate_impl(g, 0, n_events, chunk_events, seed, iteration, fid, precision, (void*)st, nullptr);
    if (rc) return rc;
    rc = vegas_reduce(g, (void*)st);
    if (rc) return rc;
    CUDA_TRY(g, vegas::launch_finalize(g->d_totals, (double)n_events, d_result, st));
    g->launches++;
    if (alpha >= 0.0) {
        CUDA_TRY(g, vegas::launch_refine(g->d_edges, g->d_totals + 4, g->dim, g->n_bins, alpha, g->d_status, st));
        g->launches++;
    }
    return VEGAS_OK;
}

int accumulate_impl(vegas_grid* g, uint64_t first_event, uint64_t count, uint64_t chunk_events, uint64_t seed,
                    uint32_t iteration, int fid, int precision, void* cuda_stream, const Tail* tail) {
    if (!check_call(g, fid, precision)) return VEGAS_EINVAL;
    if (g->active_blocks <= 0) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    const bool rot = use_rot_path(g, fid, precision);
    LaunchShape s{};
    RotShape rs{};
    vegas::IterArgs a{};
    vegas::RotArgs ra{};
    if (rot) {
        rs = rot_shape(g, fid);
        if (rs.blocks > g->active_blocks) return VEGAS_EINVAL;
        ra.edges = g->d_edges;
        ra.partials = g->d_partials;
        for (int r = 0; r < 10; ++r) {                            // C1 key schedule
            ra.k0[r] = (uint32_t)(seed & 0xFFFFFFFFu) + (uint32_t)r * 0x9E3779B9u;
            ra.k1[r] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
        }
        ra.iteration = iteration;
        ra.n_bins = g->n_bins;
        ra.n_groups = rs.n_groups;
        ra.ring = rs.ring;
        rot_constants(g, fid, precision, ra.shift, ra.scale, &ra.post_scale, &ra.fin0, &ra.fin1, &ra.jac_init, ra.fpar,
                      vegas::rot_word_map(precision == VEGAS_FP64 ? 64 : 32, g->dim), g->variant);
        if (fid == VEGAS_F_USER && g->n_obs > 0) {
            ra.obs = g->d_obs;
            ra.n_obs = g->n_obs;
            ra.obs_lo = g->obs_lo;
            ra.obs_inv_width = (double)g->n_obs / (g->obs_hi - g->obs_lo);
        }
    } else {
        if (resolve_launch(g, precision, &s)) return VEGAS_EINVAL;
        if (s.blocks > g->active_blocks) return VEGAS_EINVAL;
        a.edges = g->d_edges;
        a.partials = g->d_partials;
        a.key0 = (uint32_t)(seed & 0xFFFFFFFFu);
        a.key1 = (uint32_t)(seed >> 32);
        a.iteration = iteration;
        a.dim = g->dim;
        a.n_bins = g->n_bins;
        a.log_ct = ilog2(s.ct);
        a.log_ch = ilog2(s.ch);
        a.jac_scale = jac_scale_for(g, precision);
        if (fid != VEGAS_F_BW_POLY) {
            double fpar_unused[vegas::kRotParams];
            rot_constants(g, fid, precision, a.shift, a.scale, &a.post_scale, &a.fin0, &a.fin1, &a.jac_init, fpar_unused, false);
        }
    }
    // The fast path runs the chunk loop inside the kernel (one launch per accumulate call: the grid finishes a chunk
    // before it starts the next); the generic kernel is launched once per chunk.
    const uint64_t chunk = (chunk_events && !rot) ? chunk_events : count;
    ra.chunk = chunk_events;
    for (uint64_t done = 0, n_launch = 0; done < count; done += n_launch) {
        n_launch = (count - done < chunk) ? count - done : chunk;
        if (rot) {
            // a fast-path launch never crosses a multiple of 2^32 in the global event index: the high counter word
            // (C2) is then uniform over the launch and everything Philox derives from it alone is loop-invariant
            const uint64_t to_boundary = 0x100000000ull - ((first_event + done) & 0xFFFFFFFFull);
            if (n_launch > to_boundary) n_launch = to_boundary;
            if (n_launch > 0xFFF00000ull) n_launch = 0xFFF00000ull;     // the kernel's 32-bit event offset (+ one padded pass)
        }
        a.first_event = ra.first_event = first_event + done;
        a.count = ra.count = n_launch;
        ra.pdl = (done > 0 && !g->profiling) ? 1 : 0;   // chunk k > 0 follows chunk k-1 of this call directly in the stream
        if (tail) {                                     // the whole iteration is this one launch (one_launch_iteration)
            ra.overwrite = 1;
            ra.tail = 1;
            ra.tail_n = tail->n_events;
            ra.tail_alpha = tail->alpha;
            ra.totals = g->d_totals;
            ra.result = tail->d_result;
            ra.status = g->d_status;
            ra.counter = g->d_counter;
            ra.slices = g->d_slices;
            ra.tail_smem_doubles = (unsigned int)(rs.shmem / sizeof(double));
        }
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (g->profiling) {
            if (g->events_used + 2 > g->events.size()) {
                cudaEvent_t n0, n1;
                CUDA_TRY(g, cudaEventCreate(&n0));
                CUDA_TRY(g, cudaEventCreate(&n1));
                g->events.push_back(n0);
                g->events.push_back(n1);
            }
            e0 = g->events[g->events_used];
            e1 = g->events[g->events_used + 1];
            g->events_used += 2;
            CUDA_TRY(g, cudaEventRecord(e0, st));
        }
        if (rot)
            CUDA_TRY(g, launch_rot(g, fid, precision, g->dim, ra, rs, st));
        else
            CUDA_TRY(g, vegas::launch_iterate(fid, precision, a, g->derived[fid], s.blocks, s.threads, s.shmem, st));
        if (g->profiling) CUDA_TRY(g, cudaEventRecord(e1, st));
        g->iterate_launches++;
        g->launches++;
    }
    return VEGAS_OK;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

int vegas_reduce(vegas_grid* g, void* cuda_stream) {
    if (!g || g->active_blocks <= 0) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    const int ntot = 4 + g->dim * g->n_bins;
    CUDA_TRY(g, vegas::launch_reduce(g->d_partials, g->active_blocks, ntot, g->d_totals, st));
    g->launches++;
    return VEGAS_OK;
}

int vegas_finalize(vegas_grid* g, uint64_t n_events_total, void* cuda_stream, double* I, double* sigma,
                   double* hist_host) {
    if (!g || n_events_total < 2) return VEGAS_EINVAL;
    CUDA_TRY(g, cudaSetDevice(g->device));
    return finish_iteration(g, n_events_total, (cudaStream_t)cuda_stream, I, sigma, hist_host);
}

int vegas_finish_sharded(vegas_grid* g, uint64_t n_events_total, double alpha, void* cuda_stream, double* I, double* sigma,
                         double* hist_host) {
    if (!g || n_events_total < 2 || alpha != alpha || std::isinf(alpha)) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    CUDA_TRY(g, vegas::launch_finalize(g->d_totals, (double)n_events_total, g->d_result, st));
    g->launches++;
    const bool refine = alpha >= 0.0;
    if (refine) {
        CUDA_TRY(g, cudaMemsetAsync(g->d_status, 0, sizeof(int), st));
        CUDA_TRY(g, vegas::launch_refine(g->d_edges, g->d_totals + 4, g->dim, g->n_bins, alpha, g->d_status, st));
        g->launches++;
    }
    // { I, sigma, status }, the refinement's status word and the histogram: one synchronisation for all of them
    if (!g->h_pinned) CUDA_TRY(g, cudaHostAlloc((void**)&g->h_pinned, sizeof(double) * ((size_t)kResultStride * kMaxIter + 1), cudaHostAllocDefault));
    double* res = g->h_pinned;
    int* status_p = reinterpret_cast<int*>(g->h_pinned + (size_t)kResultStride * kMaxIter);
    *status_p = 0;
    CUDA_TRY(g, cudaMemcpyAsync(res, g->d_result, sizeof(double) * 3, cudaMemcpyDeviceToHost, st));
    if (refine) CUDA_TRY(g, cudaMemcpyAsync(status_p, g->d_status, sizeof(int), cudaMemcpyDeviceToHost, st));
    if (hist_host)
        CUDA_TRY(g, cudaMemcpyAsync(hist_host, g->d_totals + 4, sizeof(double) * (size_t)g->dim * g->n_bins, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    if (I) *I = res[0];
    if (sigma) *sigma = res[1];
    return (res[2] == 0.0 && *status_p == 0) ? VEGAS_OK : VEGAS_ENUMERIC;
}

void* vegas_totals_device(vegas_grid* g) { return g ? (void*)g->d_totals : nullptr; }
size_t vegas_totals_count(const vegas_grid* g) { return g ? 4 + (size_t)g->dim * g->n_bins : 0; }

int vegas_iterate(vegas_grid* g, uint64_t n_events, uint64_t chunk_events, uint64_t seed, uint32_t iteration,
                  int fid, int precision, void* cuda_stream, double* I, double* sigma, double* hist_host) {
    if (!check_call(g, fid, precision) || n_events < 2) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    const int rc = enqueue_iteration(g, n_events, chunk_events, seed, iteration, fid, precision, st, -1.0, g->d_result);
    if (rc) return rc;
    return fetch_result(g, st, I, sigma, hist_host);
}

int vegas_refine(vegas_grid* g, const double* hist_host, double alpha, void* cuda_stream) {
    if (!g || !(alpha >= 0.0) || !std::isfinite(alpha)) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    const double* hist = g->d_totals + 4;
    if (hist_host) {
        CUDA_TRY(g, cudaMemcpyAsync(g->d_hist_up, hist_host, sizeof(double) * g->dim * g->n_bins, cudaMemcpyHostToDevice, st));
        hist = g->d_hist_up;
    }
    CUDA_TRY(g, cudaMemsetAsync(g->d_status, 0, sizeof(int), st));
    CUDA_TRY(g, vegas::launch_refine(g->d_edges, hist, g->dim, g->n_bins, alpha, g->d_status, st));
    g->launches++;
    int status = 0;
    CUDA_TRY(g, cudaMemcpyAsync(&status, g->d_status, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    return status == 0 ? VEGAS_OK : VEGAS_ENUMERIC;
}

int vegas_combine(int n_iter, int n_skip, const double* I_k, const double* sigma_k, double* I, double* sigma,
                  double* chi2_dof) {
    if (n_iter < 1 || n_skip < 0 || n_skip >= n_iter || !I_k || !sigma_k || !I || !sigma || !chi2_dof)
        return VEGAS_EINVAL;
    const int K = n_iter - n_skip;
    bool any_zero = false;
    for (int k = n_skip; k < n_iter; ++k) {
        if (!std::isfinite(I_k[k]) || !std::isfinite(sigma_k[k]) || sigma_k[k] < 0.0) {
            // an iteration that ended in VEGAS_ENUMERIC: nothing sensible can be combined
            *I = *sigma = *chi2_dof = std::nan("");
            return VEGAS_ENUMERIC;
        }
        if (sigma_k[k] == 0.0) any_zero = true;
    }
    if (any_zero) {
        double acc = 0.0;
        for (int k = n_skip; k < n_iter; ++k) acc += I_k[k];
        *I = acc / K;
        *sigma = 0.0;
        *chi2_dof = 0.0;
        return VEGAS_OK;
    }
    // weights relative to the smallest sigma keep 1/sigma^2 in range
    double smin = sigma_k[n_skip];
    for (int k = n_skip; k < n_iter; ++k) smin = std::fmin(smin, sigma_k[k]);
    double W = 0.0, WI = 0.0;
    for (int k = n_skip; k < n_iter; ++k) {
        const double r = smin / sigma_k[k], w = r * r;
        W += w;
        WI += w * I_k[k];
    }
    const double mean = WI / W;
    double chi2 = 0.0;
    for (int k = n_skip; k < n_iter; ++k) {
        const double dev = (I_k[k] - mean) / sigma_k[k];
        chi2 += dev * dev;
    }
    *I = mean;
    *sigma = smin / std::sqrt(W);
    *chi2_dof = K > 1 ? chi2 / (K - 1) : 0.0;
    return VEGAS_OK;
}

int vegas_integrate(vegas_grid* g, int n_iter, int n_skip, uint64_t n_events, uint64_t chunk_events, uint64_t seed,
                    double alpha, int fid, int precision, void* cuda_stream, double* I, double* sigma,
                    double* chi2_dof, double* per_iter_host) {
    return vegas_integrate_from(g, 0, n_iter, n_skip, n_events, chunk_events, seed, alpha, fid, precision, cuda_stream,
                                I, sigma, chi2_dof, per_iter_host);
}

int vegas_integrate_from(vegas_grid* g, uint32_t first_iteration, int n_iter, int n_skip, uint64_t n_events,
                         uint64_t chunk_events, uint64_t seed, double alpha, int fid, int precision, void* cuda_stream,
                         double* I, double* sigma, double* chi2_dof, double* per_iter_host) {
    if (!check_call(g, fid, precision) || n_events < 2) return VEGAS_EINVAL;
    if ((uint64_t)first_iteration + (uint64_t)(n_iter > 0 ? n_iter : 0) > 0xFFFFFFFFull) return VEGAS_EINVAL;   // C2: 0xFFFFFFFF is reserved
    if (n_iter < 1 || n_iter > kMaxIter || n_skip < 0 || n_skip >= n_iter || !I || !sigma || !chi2_dof)
        return VEGAS_EINVAL;
    if (alpha != alpha || std::isinf(alpha)) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    CUDA_TRY(g, cudaMemsetAsync(g->d_status, 0, sizeof(int), st));
    // the CTAs-done tickets of the one-launch iteration reset themselves in the tail; a launch that aborted would
    // leave them counting, and only vegas_create zeroes them otherwise
    CUDA_TRY(g, cudaMemsetAsync(g->d_counter, 0, sizeof(unsigned int) * (vegas::kReduceSlices + 1), st));
    for (int k = 0; k < n_iter; ++k) {
        const int rc = enqueue_iteration(g, n_events, chunk_events, seed, first_iteration + (uint32_t)k, fid, precision, st,
                                         alpha >= 0.0 ? alpha : -1.0, g->d_result + (size_t)kResultStride * k);
        if (rc) return rc;
    }
    if (!g->h_pinned) CUDA_TRY(g, cudaHostAlloc((void**)&g->h_pinned, sizeof(double) * ((size_t)kResultStride * kMaxIter + 1), cudaHostAllocDefault));
    double* res = g->h_pinned;
    int* status_p = reinterpret_cast<int*>(g->h_pinned + (size_t)kResultStride * kMaxIter);
    CUDA_TRY(g, cudaMemcpyAsync(res, g->d_result, sizeof(double) * (size_t)kResultStride * n_iter, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaMemcpyAsync(status_p, g->d_status, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    const int status = *status_p;
    std::vector<double> Ik(n_iter), sk(n_iter);
    int rc = status == 0 ? VEGAS_OK : VEGAS_ENUMERIC;
    for (int k = 0; k < n_iter; ++k) {
        Ik[k] = res[(size_t)kResultStride * k];
        sk[k] = res[(size_t)kResultStride * k + 1];
        if (res[(size_t)kResultStride * k + 2] != 0.0) rc = VEGAS_ENUMERIC;
        if (per_iter_host) { per_iter_host[2 * k] = Ik[k]; per_iter_host[2 * k + 1] = sk[k]; }
    }
    const int rc2 = vegas_combine(n_iter, n_skip, Ik.data(), sk.data(), I, sigma, chi2_dof);
    return rc2 ? rc2 : rc;
}

size_t vegas_debug_scratch_bytes(int dim, uint32_t count) {
    if (dim < 1 || dim > VEGAS_MAX_DIM) return 0;
    const size_t per_dim = (size_t)count * dim;
    return align_up(per_dim * 4) + align_up(per_dim * 4) + align_up(per_dim * 8) + align_up((size_t)count * 8);
}

int vegas_debug_sample(vegas_grid* g, uint64_t first_event, uint32_t count, uint64_t seed, uint32_t iteration,
                       int fid, int precision, void* dev_scratch, void* cuda_stream, uint32_t* words,
                       int32_t* bins, double* x, double* fJ) {
    if (!check_call(g, fid, precision) || fid == VEGAS_F_USER || !dev_scratch || count == 0) return VEGAS_EINVAL;
    if (((uintptr_t)dev_scratch) % kAlign) return VEGAS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(g, cudaSetDevice(g->device));
    const size_t per_dim = (size_t)count * g->dim;
    unsigned char* base = (unsigned char*)dev_scratch;
    vegas::DebugArgs a{};
    a.edges = g->d_edges;
    a.first_event = first_event;
    a.count = count;
    a.key0 = (uint32_t)(seed & 0xFFFFFFFFu);
    a.key1 = (uint32_t)(seed >> 32);
    a.iteration = iteration;
    a.dim = g->dim;
    a.n_bins = g->n_bins;
    a.jac_scale = jac_scale_for(g, precision);
    a.words = (uint32_t*)base;                 base += align_up(per_dim * 4);
    a.bins = (int32_t*)base;                   base += align_up(per_dim * 4);
    a.x = (double*)base;                       base += align_up(per_dim * 8);
    a.fJ = (double*)base;
    // both K1 kernels form u_j, f and v through the affine map for every integrand but BW_POLY beyond the fast path
    const bool rot = fid != VEGAS_F_BW_POLY || use_rot_path(g, fid, precision);
    a.word_map = rot && vegas::rot_word_map(precision == VEGAS_FP64 ? 64 : 32, g->dim);
    a.variant = g->variant;
    if (rot) rot_constants(g, fid, precision, a.shift, a.scale, &a.post_scale, &a.fin0, &a.fin1, &a.jac_init, a.fpar, a.word_map != 0, g->variant);
    CUDA_TRY(g, vegas::launch_debug(fid, precision, rot, a, g->derived[fid], st));
    g->launches++;
    if (words) CUDA_TRY(g, cudaMemcpyAsync(words, a.words, per_dim * 4, cudaMemcpyDeviceToHost, st));
    if (bins) CUDA_TRY(g, cudaMemcpyAsync(bins, a.bins, per_dim * 4, cudaMemcpyDeviceToHost, st));
    if (x) CUDA_TRY(g, cudaMemcpyAsync(x, a.x, per_dim * 8, cudaMemcpyDeviceToHost, st));
    if (fJ) CUDA_TRY(g, cudaMemcpyAsync(fJ, a.fJ, (size_t)count * 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(g, cudaStreamSynchronize(st));
    return VEGAS_OK;
}

static size_t callback_slot_bytes(int dim, uint32_t batch_events) {
    return vegas_debug_scratch_bytes(dim, batch_events) + align_up((size_t)batch_events * 8);
}

// two slots: the device samples batch k+1 (and copies its points to the host) while the host evaluates batch k
size_t vegas_callback_scratch_bytes(int dim, uint32_t batch_events) {
    if (dim < 1 || dim > VEGAS_MAX_DIM || batch_events == 0) return 0;
    return 2 * callback_slot_bytes(dim, batch_events);
}

int vegas_iterate_callback(vegas_grid* g, uint64_t n_events, uint32_t batch_events, uint64_t seed, uint32_t iteration,
                           vegas_host_integrand fn, void* user, void* dev_scratch, size_t scratch_bytes,
                           void* cuda_stream, double* I, double* sigma, double* hist_host) {
    if (!g || !fn || !dev_scratch || n_events < 2 || batch_events == 0) return VEGAS_EINVAL;
    if (((uintptr_t)dev_scratch) % kAlign) return VEGAS_EINVAL;
    const size_t slot_bytes = callback_slot_bytes(g->dim, batch_events);
    if (scratch_bytes < slot_bytes) return VEGAS_EINVAL;
    const int n_slots = scratch_bytes >= 2 * slot_bytes ? 2 : 1;      // one slot: the strictly serial form
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = vegas_begin_iteration(g, cuda_stream);
    if (rc) return rc;
    const int dim = g->dim;
    const size_t per_dim = (size_t)batch_events * dim;
    // page-locked host staging (x and f per slot), kept with the grid and grown on demand; four events
    const size_t need = 2 * (per_dim + batch_events);
    if (g->h_cb_doubles < need) {
        if (g->h_cb) cudaFreeHost(g->h_cb);
        g->h_cb = nullptr;
        g->h_cb_doubles = 0;
        CUDA_TRY(g, cudaHostAlloc((void**)&g->h_cb, sizeof(double) * need, cudaHostAllocDefault));
        g->h_cb_doubles = need;
    }
    for (cudaEvent_t& ev : g->cb_ev)
        if (!ev) CUDA_TRY(g, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    vegas::DebugArgs a[2];
    double* d_f[2];
    double* x_host[2];
    double* f_host[2];
    for (int s = 0; s < 2; ++s) {
        unsigned char* base = (unsigned char*)dev_scratch + (s < n_slots ? (size_t)s * slot_bytes : 0);
        a[s] = vegas::DebugArgs{};
        a[s].edges = g->d_edges;
        a[s].key0 = (uint32_t)(seed & 0xFFFFFFFFu);
        a[s].key1 = (uint32_t)(seed >> 32);
        a[s].iteration = iteration;
        a[s].dim = dim;
        a[s].n_bins = g->n_bins;
        a[s].jac_scale = jac_scale_for(g, VEGAS_FP64);
        a[s].words = (uint32_t*)base;                 base += align_up(per_dim * 4);
        a[s].bins = (int32_t*)base;                   base += align_up(per_dim * 4);
        a[s].x = (double*)base;                       base += align_up(per_dim * 8);
        a[s].fJ = (double*)base;                      base += align_up((size_t)batch_events * 8);
        d_f[s] = (double*)base;
        x_host[s] = g->h_cb + (size_t)s * (per_dim + batch_events);
        f_host[s] = x_host[s] + per_dim;
    }
    const int blocks = g->active_blocks < g->sm_count ? g->active_blocks : g->sm_count;
    const uint64_t n_batches = (n_events + batch_events - 1) / batch_events;
    auto batch_size = [&](uint64_t k) {
        const uint64_t done = k * (uint64_t)batch_events;
        return (uint32_t)((n_events - done < batch_events) ? n_events - done : batch_events);
    };
    // S1-S3 for batch k with f = 1: x, bins and J = prod n_bins Delta go to the slot's scratch (the only place in the
    // library where per-event arrays exist), x on to the host
    auto enqueue_sample = [&](uint64_t k, int s) -> int {
        a[s].first_event = k * (uint64_t)batch_events;
        a[s].count = batch_size(k);
        CUDA_TRY(g, vegas::launch_debug(VEGAS_F_CONST, VEGAS_FP64, false, a[s], g->derived[VEGAS_F_CONST], st));
        CUDA_TRY(g, cudaMemcpyAsync(x_host[s], a[s].x, sizeof(double) * (size_t)a[s].count * dim, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(g, cudaEventRecord(g->cb_ev[s], st));
        g->launches++;
        return VEGAS_OK;
    };
    // the two-slot pipeline; on any error the caller's stream is drained before returning (below): copies into the
    // page-locked staging and kernels on the scratch slots may still be in flight, and the next call may free both
    auto pipeline = [&]() -> int {
    int rc = enqueue_sample(0, 0);
    if (rc) return rc;
    bool f_in_flight[2] = {false, false};
    for (uint64_t k = 0; k < n_batches; ++k) {
        const int s = n_slots == 2 ? (int)(k & 1) : 0;
        const uint32_t n = batch_size(k);
        if (n_slots == 2 && k + 1 < n_batches) {           // the device goes on with batch k+1 while the host evaluates batch k
            rc = enqueue_sample(k + 1, s ^ 1);
            if (rc) return rc;
        }
        CUDA_TRY(g, cudaEventSynchronize(g->cb_ev[s]));                               // x of batch k is on the host
        if (f_in_flight[s]) CUDA_TRY(g, cudaEventSynchronize(g->cb_ev[2 + s]));       // f of batch k-2 has left f_host[s]
        fn(x_host[s], (uint64_t)n, dim, f_host[s], user);                             // S4 on the host
        CUDA_TRY(g, cudaMemcpyAsync(d_f[s], f_host[s], sizeof(double) * n, cudaMemcpyHostToDevice, st));
        CUDA_TRY(g, cudaEventRecord(g->cb_ev[2 + s], st));
        f_in_flight[s] = true;
        CUDA_TRY(g, vegas::launch_accumulate_batch(d_f[s], a[s].fJ, a[s].bins, n, dim, g->n_bins, g->d_partials, blocks, st));
        g->launches++;
        if (n_slots == 1 && k + 1 < n_batches) {           // one slot: the next sample overwrites what accumulate reads -- stream order
            rc = enqueue_sample(k + 1, 0);
            if (rc) return rc;
        }
    }
    return vegas_reduce(g, cuda_stream);
    };
    rc = pipeline();
    if (rc) {
        cudaStreamSynchronize(st);                          // nothing of this call is left in flight
        return rc;
    }
    return finish_iteration(g, n_events, st, I, sigma, hist_host);
}

int vegas_set_launch(vegas_grid* g, int blocks, int threads, int table_copies, int hist_copies) {
    if (!g || blocks < 0 || threads < 0 || table_copies < 0 || hist_copies < 0) return VEGAS_EINVAL;
    auto pow2 = [](int v) { return v == 0 || (v & (v - 1)) == 0; };
    if (!pow2(table_copies) || !pow2(hist_copies) || table_copies > 32 || hist_copies > 32) return VEGAS_EINVAL;
    vegas_grid trial = *g;
    trial.events.clear();
    trial.cfg_blocks = blocks;
    trial.cfg_threads = threads;
    trial.cfg_ct = table_copies;
    trial.cfg_ch = hist_copies;
    LaunchShape s;
    if (resolve_launch(&trial, VEGAS_FP64, &s) || resolve_launch(&trial, VEGAS_FP32, &s)) return VEGAS_EINVAL;
    g->cfg_blocks = blocks;
    g->cfg_threads = threads;
    g->cfg_ct = table_copies;
    g->cfg_ch = hist_copies;
    g->active_blocks = 0;
    return VEGAS_OK;
}

int vegas_set_variant(vegas_grid* g, int variant) {
    if (!g || (variant != VEGAS_VARIANT_NONE && variant != VEGAS_VARIANT_U53 && variant != VEGAS_VARIANT_Q32)) return VEGAS_EINVAL;
    g->variant = variant;
    return VEGAS_OK;
}

int vegas_get_variant(const vegas_grid* g) { return g ? g->variant : VEGAS_EINVAL; }

int vegas_get_launch(vegas_grid* g, int integrand_id, int precision, int* path, int* blocks, int* threads,
                     int* table_copies, int* hist_copies, size_t* shared_bytes) {
    if (!g || (precision != VEGAS_FP64 && precision != VEGAS_FP32) || integrand_id < 0 || integrand_id > VEGAS_F_GENZ_DISCONTINUOUS)
        return VEGAS_EINVAL;
    if (use_rot_path(g, integrand_id, precision)) {
        const RotShape r = rot_shape(g, integrand_id);
        if (blocks) *blocks = r.blocks;
        if (threads) *threads = r.threads;
        if (table_copies) *table_copies = precision == VEGAS_FP64 ? 2 : 4;
        if (hist_copies) *hist_copies = 8 * r.n_groups;
        if (shared_bytes) *shared_bytes = r.shmem;
        if (path) *path = 1;
        return VEGAS_OK;
    }
    LaunchShape s;
    if (resolve_launch(g, precision, &s)) return VEGAS_EINVAL;
    if (blocks) *blocks = s.blocks;
    if (threads) *threads = s.threads;
    if (table_copies) *table_copies = s.ct;
    if (hist_copies) *hist_copies = s.ch;
    if (shared_bytes) *shared_bytes = s.shmem;
    if (path) *path = 0;
    return VEGAS_OK;
}

int vegas_set_profiling(vegas_grid* g, int on) {
    if (!g) return VEGAS_EINVAL;
    g->profiling = on != 0;
    return VEGAS_OK;
}

int vegas_kernel_time_ms(vegas_grid* g, double* iterate_kernel_ms, uint64_t* iterate_launches) {
    if (!g) return VEGAS_EINVAL;
    CUDA_TRY(g, cudaSetDevice(g->device));
    for (size_t i = 0; i + 1 < g->events_used; i += 2) {
        CUDA_TRY(g, cudaEventSynchronize(g->events[i + 1]));
        float ms = 0.f;
        CUDA_TRY(g, cudaEventElapsedTime(&ms, g->events[i], g->events[i + 1]));
        g->kernel_ms_acc += (double)ms;
    }
    g->events_used = 0;
    if (iterate_kernel_ms) *iterate_kernel_ms = g->kernel_ms_acc;
    if (iterate_launches) *iterate_launches = g->iterate_launches;
    return VEGAS_OK;
}

uint64_t vegas_launch_count(const vegas_grid* g) { return g ? g->launches : 0; }

int vegas_reset_counters(vegas_grid* g) {
    if (!g) return VEGAS_EINVAL;
    g->events_used = 0;
    g->kernel_ms_acc = 0.0;
    g->iterate_launches = 0;
    g->launches = 0;
    return VEGAS_OK;
}

}  // extern "C"
#pragma GCC visibility pop

// =============================================================================================
// vegas_iterate_static: one iteration for a caller that cannot give the library any device memory beyond its inputs
// and outputs (include/vegas.h says who that is).  The working memory of the generic fused kernel K1 and of the
// reduction K2 -- one row { S1 hi, S1 lo, S2 hi, S2 lo, H[dim][n_bins] } per CTA, then one row of totals -- lives in
// the array below instead of a caller workspace.  Nothing in this path allocates: no cudaMalloc / cudaFree /
// cudaMallocHost, no vegas_grid with a workspace; the kernels and their launchers are the ones vegas_iterate uses
// with pinned copy counts, given pointers into this array.
//
// The array is device memory that the CUDA runtime reserves on every GPU where this translation unit's device code
// gets loaded, until the process exits (kStaticDoubles * 8 = 2 642 976 bytes).  On the host the name
// g_static_scratch is only a handle for the runtime's symbol table, NOT an address a kernel can use: the device
// address is asked for once per device with cudaGetSymbolAddress (static_setup) and that pointer is what the
// kernels get.
// =============================================================================================
namespace {
constexpr int kStaticMaxBlocks = 160;                                        // >= one CTA per SM of a B200 (148)
constexpr size_t kStaticRow = 4 + (size_t)VEGAS_STATIC_MAX_ENTRIES;          // doubles per CTA row / totals row
constexpr size_t kStaticDoubles = kStaticRow * (kStaticMaxBlocks + 1);       // CTA rows, then the totals row
}  // namespace

static __device__ __align__(256) double g_static_scratch[kStaticDoubles];

namespace {

struct StaticDevice {
    bool ready = false;
    double* scratch = nullptr;      // DEVICE address of g_static_scratch on this GPU
    int sm_count = 0;
    size_t smem_optin = 0;
};
StaticDevice g_static_dev[vegas::kMaxDevices];
std::mutex g_static_mutex;

// Once per device, with that device current: the array's device address and the limits the launch shape needs.
cudaError_t static_setup(int dev, StaticDevice* out) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& d = g_static_dev[dev];
    if (!d.ready) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        if (e != cudaSuccess) return e;
        int sms = 0, optin = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return e;
        d.scratch = static_cast<double*>(ptr);
        d.sm_count = sms;
        d.smem_optin = (size_t)optin;
        d.ready = true;
    }
    *out = d;
    return cudaSuccess;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

int vegas_iterate_static(const double* edges_dev, int dim, int n_bins, uint64_t n_events, uint64_t seed,
                         uint32_t iteration, int fid, const double* params_host, int n_params, int precision,
                         void* cuda_stream, double* result_dev, double* hist_dev) {
    if (!edges_dev || !result_dev || n_events < 2 || !valid_shape(dim, n_bins)) return VEGAS_EINVAL;
    if ((size_t)dim * n_bins > (size_t)VEGAS_STATIC_MAX_ENTRIES) return VEGAS_ELIMIT;      // before anything is launched
    if (fid == VEGAS_F_USER) return VEGAS_EINVAL;

    // a host-only grid object: it carries the shape and the derived integrand parameters through the same
    // validation and derivation as vegas_set_params / vegas_accumulate; it has no workspace and owns nothing
    vegas_grid host;
    host.dim = dim;
    host.n_bins = n_bins;
    int rc = vegas_set_params(&host, fid, params_host, n_params);
    if (rc) return rc;
    if (!check_call(&host, fid, precision)) return VEGAS_EINVAL;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= vegas::kMaxDevices) return VEGAS_ECUDA;
    StaticDevice sd;
    if (static_setup(dev, &sd) != cudaSuccess) return VEGAS_ECUDA;
    host.device = dev;
    host.sm_count = sd.sm_count;
    host.smem_optin = sd.smem_optin;
    host.cfg_blocks = sd.sm_count < kStaticMaxBlocks ? sd.sm_count : kStaticMaxBlocks;     // one CTA per SM, rows permitting
    LaunchShape s;
    if (resolve_launch(&host, precision, &s)) return VEGAS_EINVAL;

    const size_t nent = (size_t)dim * n_bins, ntot = 4 + nent;
    double* partials = sd.scratch;                            // [s.blocks][ntot]
    double* totals = sd.scratch + (size_t)kStaticMaxBlocks * kStaticRow;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    vegas::IterArgs a{};
    a.edges = edges_dev;
    a.partials = partials;
    a.first_event = 0;
    a.count = n_events;
    a.key0 = (uint32_t)(seed & 0xFFFFFFFFu);
    a.key1 = (uint32_t)(seed >> 32);
    a.iteration = iteration;
    a.dim = dim;
    a.n_bins = n_bins;
    a.log_ct = ilog2(s.ct);
    a.log_ch = ilog2(s.ch);
    a.jac_scale = jac_scale_for(&host, precision);
    if (fid != VEGAS_F_BW_POLY) {
        double fpar_unused[vegas::kRotParams];
        rot_constants(&host, fid, precision, a.shift, a.scale, &a.post_scale, &a.fin0, &a.fin1, &a.jac_init, fpar_unused, false);
    }
    // the CTA rows are accumulated into (K1 adds to its row): the previous call's sums must go first, in stream order
    CUDA_TRY(nullptr, cudaMemsetAsync(partials, 0, sizeof(double) * ntot * s.blocks, st));
    CUDA_TRY(nullptr, vegas::launch_iterate(fid, precision, a, host.derived[fid], s.blocks, s.threads, s.shmem, st));
    CUDA_TRY(nullptr, vegas::launch_reduce(partials, s.blocks, (int)ntot, totals, st));     // writes every total
    CUDA_TRY(nullptr, vegas::launch_finalize(totals, (double)n_events, result_dev, st));
    if (hist_dev)
        CUDA_TRY(nullptr, cudaMemcpyAsync(hist_dev, totals + 4, sizeof(double) * nent, cudaMemcpyDeviceToDevice, st));
    return VEGAS_OK;
}

const char* vegas_strerror(int code) {
    switch (code) {
    case VEGAS_OK: return "ok";
    case VEGAS_EINVAL: return "invalid argument";
    case VEGAS_ECUDA: return "CUDA runtime or launch failure (see vegas_last_cuda_error)";
    case VEGAS_ENUMERIC: return "non-finite sums, or a histogram row without a finite positive sum in refine";
    case VEGAS_ELIMIT: return "vegas_iterate_static: dim * n_bins exceeds VEGAS_STATIC_MAX_ENTRIES (2048), the shape its built-in scratch holds; use a vegas_grid";
    default: return "unknown error code";
    }
}

const char* vegas_last_cuda_error(const vegas_grid* g) { return g ? g->cuda_err : ""; }

const char* vegas_version(void) { return "vegas_b200 0.1 sm_100a"; }

}  // extern "C"
#pragma GCC visibility pop
