// vegas_kernels.cu -- the sm_100a kernels of the Vegas iteration library and their launchers.
//   K1 k_iterate   fused RNG -> split -> grid map -> integrand -> S1, S2, histogram   (S1..S6)
//   K2 k_reduce    deterministic second-level reduction over the per-CTA partials
//      k_finalize  I = S1/n, sigma^2 = (S2/n - I^2)/(n-1) in double-double             (S7)
//   K3 k_refine    smooth, normalise, compress with alpha, rebin; one CTA per dimension (S8)
//   K4 k_debug     parity hook: words, bins, x, f*J of single events through K1's device functions
// Step names S1..S9 are SURVEY.md 8(a); readings C1..C11 are DESIGN.md.
#include "vegas_kernels.h"

#include <mutex>

#include "vegas_device.cuh"
#include "vegas_iterate_rot.cuh"

namespace vegas {

// The small kernels that follow the fused kernel in the stream (K2, finalize, K3) are launched with programmatic
// stream serialisation: their launch overlaps the tail of the kernel before them, and they wait here for it to
// complete before they read anything.  A no-op when the kernel was launched the ordinary way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t shmem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = shmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

template <typename T> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };

// One grid-table entry from two master-grid edges (C4).  fp64: (X_b, Delta).  fp32 (C11):
// (X_b, n_bins*Delta) rounded to fp32 -- the per-dimension Jacobian factor itself, so that the
// running product stays O(1) instead of underflowing like prod Delta would in fp32.
template <typename T>
__device__ __forceinline__ typename Vec2<T>::type make_entry(double x0, double x1, int n_bins);
template <>
__device__ __forceinline__ double2 make_entry<double>(double x0, double x1, int) {
    return make_double2(x0, x1 - x0);
}
template <>
__device__ __forceinline__ float2 make_entry<float>(double x0, double x1, int n_bins) {
    return make_float2((float)x0, (float)((double)n_bins * (x1 - x0)));
}

// x_j and the Jacobian factor from the table entry and the low product word (C3, C4).
template <typename T> struct MapConst;
template <> struct MapConst<double> {
    __device__ __forceinline__ MapConst(int) {}
    __device__ __forceinline__ double x(double2 ent, uint32_t lo) const {
        return fma(ent.y, offset_f64(lo), ent.x);
    }
};
template <> struct MapConst<float> {
    float c24, c25;
    __device__ __forceinline__ MapConst(int n_bins)
        : c24(5.9604644775390625e-08f / (float)n_bins), c25(2.98023223876953125e-08f / (float)n_bins) {}
    __device__ __forceinline__ float x(float2 ent, uint32_t lo) const {
        return fmaf(ent.y, offset_f32_scaled(lo, c24, c25), ent.x);
    }
};

// ---------------------------------------------------------------------------------------------
// K1.  One thread = one event at a time, grid-stride over the launch's event range.
// Shared memory: the grid table, `ct` bank-interleaved copies ([entry][copy], copy = lane mod ct),
// then the histogram, `ch` bank-interleaved fp64 copies ([bin][copy], copy = lane mod ch), then the
// block-reduction scratch.  The copies put the lanes of one shared-memory wavefront on different
// banks whatever bins they drew.
// NBLK = ceil(dim/4) Philox blocks per event, compile time so that the packed bin indices
// (one byte per dimension) live in registers.
// ---------------------------------------------------------------------------------------------
// CONST, GAUSS and the product peak go through the affine variable u_j = scale_j (x_j - shift_j) exactly as on the
// fast path (table entry (A, B) with u = A + B w, IntegrandU, value()); BW_POLY (dim > 8 only gets here) keeps the
// plain map x_j = X_b + Delta r and its parameters in the constant bank.
template <int FID, typename T, int NBLK>
__global__ void __launch_bounds__(kIterMaxThreads, kIterMinBlocks)
k_iterate(const __grid_constant__ IterArgs a, const __grid_constant__ FParams<T> fp) {
    using T2 = typename Vec2<T>::type;
    constexpr bool AFF = (FID != VEGAS_F_BW_POLY);
    constexpr int NCH = AFF ? rot_chains(VEGAS_MAX_DIM, FID, sizeof(T) == 4) : 1;   // 1, or 4 for the fp32 product peak
    extern __shared__ __align__(16) unsigned char smem[];
    const int dim = a.dim, nb = a.n_bins, nent = dim * nb;
    const int ct = 1 << a.log_ct, ch = 1 << a.log_ch;
    const uint32_t table_bytes = (uint32_t)(sizeof(T2) * nent * ct);
    T2* table = reinterpret_cast<T2*>(smem);
    double* hist = reinterpret_cast<double*>(smem + table_bytes);
    dd* red = reinterpret_cast<dd*>(smem + table_bytes + (uint32_t)(8 * nent * ch));

    for (int i = threadIdx.x; i < nent; i += blockDim.x) {
        const int j = i / nb, b = i - j * nb;
        const double* X = a.edges + (size_t)j * (nb + 1);
        const T2 ent = AFF ? RotEntry<T>::make(X[b], X[b + 1], a.shift[j], a.scale[j]) : make_entry<T>(X[b], X[b + 1], nb);
        for (int c = 0; c < ct; ++c) table[i * ct + c] = ent;
    }
    for (int i = threadIdx.x; i < nent * ch; i += blockDim.x) hist[i] = 0.0;
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const unsigned char* tlane = smem + (uint32_t)(lane & (ct - 1)) * (uint32_t)sizeof(T2);
    const uint32_t tstride = (uint32_t)sizeof(T2) << a.log_ct;       // bytes per table entry row
    double* hlane = hist + (lane & (ch - 1));
    const PhiloxKey ks = philox_key_schedule(a.key0, a.key1);
    const MapConst<T> mapc(nb);
    const double jac_scale = a.jac_scale;

    double s1 = 0.0, c1 = 0.0, s2 = 0.0, c2 = 0.0;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long q = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; q < a.count;
         q += stride) {
        const unsigned long long e = a.first_event + q;
        const uint32_t e_lo = (uint32_t)e, e_hi = (uint32_t)(e >> 32);
        Integrand<FID, T> f;
        f.begin();
        IntegrandU<AFF ? FID : VEGAS_F_CONST, T, NCH> fu;
        const RotCtx<AFF ? FID : VEGAS_F_CONST, T, 1> ctx{};
        fu.begin(ctx);
        T jac[NCH];
#pragma unroll
        for (int c = 0; c < NCH; ++c) jac[c] = (c || !AFF) ? (T)1 : (T)a.jac_init;
        uint32_t packed[NBLK];
#pragma unroll
        for (int blk = 0; blk < NBLK; ++blk) {
            uint32_t w[4];
            philox4x32_10((uint32_t)blk, a.iteration, e_lo, e_hi, ks, w);
            uint32_t pk = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int j = 4 * blk + i;
                if (j < dim) {
                    uint32_t b, lo;
                    split_word(w[i], (uint32_t)nb, b, lo);
                    const T2 ent = *reinterpret_cast<const T2*>(tlane + ((uint32_t)(j * nb) + b) * tstride);
                    jac[i & (NCH - 1)] *= ent.y;
                    if (AFF) fu.dim(RotEntry<T>::u(ent, lo), 0, i, ctx);
                    else f.dim(j, mapc.x(ent, lo), fp);
                    pk |= b << (8 * i);
                }
            }
            packed[blk] = pk;
        }
        double v;
        if (!AFF) v = (double)(f.finish(fp) * jac[0]) * jac_scale;
        else if (sizeof(T) == 8) v = (double)fu.finish((T)a.fin0, (T)a.fin1) * ((double)chain_prod<NCH, T>(jac) * a.post_scale);
        else v = (double)fu.value(jac, (T)a.fin0, (T)a.fin1) * a.post_scale;          // C11: v formed in fp32, then widened
        const double v2 = v * v;
        kahan_add(s1, c1, v);
        kahan_add(s2, c2, v2);
#pragma unroll
        for (int blk = 0; blk < NBLK; ++blk) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int j = 4 * blk + i;
                if (j < dim) {
                    const uint32_t b = (packed[blk] >> (8 * i)) & 0xFFu;
                    atomicAdd(hlane + (((uint32_t)(j * nb) + b) << a.log_ch), v2);
                }
            }
        }
    }

    // S5: warp shuffle -> CTA -> this CTA's partial (accumulated over the launches of an iteration)
    dd t1 = dd_warp_sum(fast_two_sum(s1, -c1));
    dd t2 = dd_warp_sum(fast_two_sum(s2, -c2));
    const int warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
    if (lane == 0) { red[2 * warp] = t1; red[2 * warp + 1] = t2; }
    __syncthreads();
    double* part = a.partials + (size_t)blockIdx.x * (4 + nent);
    if (warp == 0) {
        t1 = (lane < nwarps) ? red[2 * lane] : dd{0.0, 0.0};
        t2 = (lane < nwarps) ? red[2 * lane + 1] : dd{0.0, 0.0};
        t1 = dd_warp_sum(t1);
        t2 = dd_warp_sum(t2);
        if (lane == 0) {
            t1 = dd_add(t1, dd{part[0], part[1]});
            t2 = dd_add(t2, dd{part[2], part[3]});
            part[0] = t1.hi; part[1] = t1.lo; part[2] = t2.hi; part[3] = t2.lo;
        }
    }
    // S6: merge the copies in fixed order, one coalesced pass per CTA
    for (int i = threadIdx.x; i < nent; i += blockDim.x) {
        double h = 0.0;
        for (int c = 0; c < ch; ++c) h += hist[i * ch + c];
        part[4 + i] += h;
    }
}

// ---------------------------------------------------------------------------------------------
// K2: totals[i] = sum over CTAs of partials[cta][i] in a fixed association (i >= 4: histogram, plain fp64, 8 strided
// slices of the CTAs then the slices in order; i < 4: the two double-double sums, one warp each).
// ---------------------------------------------------------------------------------------------
__global__ void k_reduce(const double* __restrict__ partials, int n_parts, int n_tot, double* __restrict__ totals) {
    pdl_wait();
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (blockIdx.x == 0) {
        if (t >= 64) return;
        reduce_dd_sum(partials, n_parts, n_tot, 2 * (t >> 5), t & 31, totals);     // S1 (warp 0) and S2 (warp 1)
        return;
    }
    // histogram totals: block b > 0 owns 32 consecutive totals; its 8 warps each add every 8th CTA's partial,
    // and warp 0 adds the 8 slice sums in slice order -- a fixed association
    __shared__ double slice[8][32];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = 4 + ((int)blockIdx.x - 1) * 32 + lane;
    slice[w][lane] = (i < n_tot) ? reduce_hist_slice(partials, n_parts, n_tot, i, w) : 0.0;
    __syncthreads();
    if (w == 0 && i < n_tot) {
        double t = slice[0][lane];
        for (int k = 1; k < 8 && k < n_parts; ++k) t += slice[k][lane];
        totals[i] = t;
    }
}

// S7 (C7), one thread
__global__ void k_finalize(const double* __restrict__ totals, double n, double* __restrict__ result) {
    pdl_wait();
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    finalize_result(totals, n, result);
}

// ---------------------------------------------------------------------------------------------
// K3 (C8): one CTA per dimension (refine_dimension in vegas_device.cuh).
// status[0] is set to VEGAS_ENUMERIC if a dimension has no finite positive smoothed sum.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(VEGAS_MAX_BINS)
k_refine(double* __restrict__ edges, const double* __restrict__ hist, int n_bins, double alpha, int* status) {
    __shared__ double scratch[refine_scratch_doubles(VEGAS_MAX_BINS)];
    pdl_wait();
    const int j = blockIdx.x;
    refine_dimension(edges + (size_t)j * (n_bins + 1), hist + (size_t)j * n_bins, n_bins, alpha, status, scratch,
                     (int)threadIdx.x, (int)blockDim.x, SyncCta{});
}

// ---------------------------------------------------------------------------------------------
// K4: one thread per event, generic in dim; same device functions as K1.
// ---------------------------------------------------------------------------------------------
template <int FID, typename T>
__global__ void k_debug(const DebugArgs a, const __grid_constant__ FParams<T> fp) {
    using T2 = typename Vec2<T>::type;
    const uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= a.count) return;
    const unsigned long long e = a.first_event + q;
    const int dim = a.dim, nb = a.n_bins;
    const PhiloxKey ks = philox_key_schedule(a.key0, a.key1);
    const MapConst<T> mapc(nb);
    Integrand<FID, T> f;
    f.begin();
    T jac = (T)1;
    uint32_t w[4] = {0, 0, 0, 0};
    for (int j = 0; j < dim; ++j) {
        if ((j & 3) == 0) philox4x32_10((uint32_t)(j >> 2), a.iteration, (uint32_t)e, (uint32_t)(e >> 32), ks, w);
        const uint32_t word = (j & 3) == 0 ? w[0] : (j & 3) == 1 ? w[1] : (j & 3) == 2 ? w[2] : w[3];
        uint32_t b, lo;
        split_word(word, (uint32_t)nb, b, lo);
        const double* X = a.edges + (size_t)j * (nb + 1);
        const T2 ent = make_entry<T>(X[b], X[b + 1], nb);
        const T x = mapc.x(ent, lo);
        jac *= ent.y;
        f.dim(j, x, fp);
        a.words[(size_t)q * dim + j] = word;
        a.bins[(size_t)q * dim + j] = (int32_t)b;
        a.x[(size_t)q * dim + j] = (double)x;
    }
    a.fJ[q] = (double)(f.finish(fp) * jac) * a.jac_scale;
}

// ---------------------------------------------------------------------------------------------
// Host-callback path (vegas_iterate_callback: integrands written in C or Fortran):
// the batch's points were produced by k_debug<CONST> (x, bins, J), the caller's host function supplied f; this kernel
// is steps S5/S6 on the stored batch.  Not the hot path: it exists so that a host integrand can be used at all.
// Shared memory: one fp64 histogram of dim*n_bins words, then the block-reduction scratch.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_accumulate_batch(const double* __restrict__ f, const double* __restrict__ J, const int32_t* __restrict__ bins,
                   uint32_t count, int dim, int nb, double* __restrict__ partials) {
    extern __shared__ __align__(16) unsigned char smem_cb[];
    const int nent = dim * nb;
    double* hist = reinterpret_cast<double*>(smem_cb);
    dd* red = reinterpret_cast<dd*>(smem_cb + sizeof(double) * nent);
    for (int i = threadIdx.x; i < nent; i += blockDim.x) hist[i] = 0.0;
    __syncthreads();
    double s1 = 0.0, c1 = 0.0, s2 = 0.0, c2 = 0.0;
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < count; e += gridDim.x * blockDim.x) {
        const double v = f[e] * J[e];                       // C6: v = f J
        const double v2 = v * v;
        kahan_add(s1, c1, v);
        kahan_add(s2, c2, v2);
        const int32_t* b = bins + (size_t)e * dim;
        for (int j = 0; j < dim; ++j) atomicAdd(hist + j * nb + b[j], v2);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
    dd t1 = dd_warp_sum(fast_two_sum(s1, -c1));
    dd t2 = dd_warp_sum(fast_two_sum(s2, -c2));
    if (lane == 0) { red[2 * warp] = t1; red[2 * warp + 1] = t2; }
    __syncthreads();
    double* part = partials + (size_t)blockIdx.x * (4 + nent);
    if (warp == 0) {
        t1 = (lane < nwarps) ? red[2 * lane] : dd{0.0, 0.0};
        t2 = (lane < nwarps) ? red[2 * lane + 1] : dd{0.0, 0.0};
        t1 = dd_warp_sum(t1);
        t2 = dd_warp_sum(t2);
        if (lane == 0) {
            t1 = dd_add(t1, dd{part[0], part[1]});
            t2 = dd_add(t2, dd{part[2], part[3]});
            part[0] = t1.hi; part[1] = t1.lo; part[2] = t2.hi; part[3] = t2.lo;
        }
    }
    for (int i = threadIdx.x; i < nent; i += blockDim.x) part[4 + i] += hist[i];
}

// K4 for the fast path: u_j and f*J through the device functions of k_iterate_rot (RotEntry,
// IntegrandU); x_j, which that kernel never forms, is reported from the plain map (C4).
template <int FID, typename T>
__global__ void k_debug_rot(const __grid_constant__ DebugArgs a) {
    using E = RotEntry<T>;
    const uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= a.count) return;
    const unsigned long long e = a.first_event + q;
    const int dim = a.dim, nb = a.n_bins;
    const PhiloxKey ks = philox_key_schedule(a.key0, a.key1);
    RotCtx<FID, T, VEGAS_MAX_DIM / 4> ctx;     // lane 0's view: gamma = 0, dimension j at (j >> 2, j & 3)
    ctx.init(a, dim, 0, 0);
    constexpr int NCH = rot_chains(VEGAS_MAX_DIM, FID, sizeof(T) == 4);     // 1, or 4 for the fp32 product peak
    IntegrandU<FID, T, NCH> f;
    f.begin(ctx);
    T jac[NCH];
    for (int c = 0; c < NCH; ++c) jac[c] = c ? (T)1 : (T)a.jac_init;
    uint32_t w[4] = {0, 0, 0, 0};
    for (int j = 0; j < dim; ++j) {
        if ((j & 3) == 0) philox4x32_10((uint32_t)(j >> 2), a.iteration, (uint32_t)e, (uint32_t)(e >> 32), ks, w);
        const uint32_t word = (j & 3) == 0 ? w[0] : (j & 3) == 1 ? w[1] : (j & 3) == 2 ? w[2] : w[3];
        uint32_t b, lo;
        split_word(word, (uint32_t)nb, b, lo);                 // for the plain map below (x is reported, not used)
        const double* X = a.edges + (size_t)j * (nb + 1);
        typename E::type ent;
        T u;
        double x_var = 0.0;
        uint32_t word_var = word;
        if (sizeof(T) == 8 && a.variant == kVarU53) {          // C3': two words per draw, block j >> 1
            uint32_t o4[4];
            philox4x32_10((uint32_t)(j >> 1), a.iteration, (uint32_t)e, (uint32_t)(e >> 32), ks, o4);
            const uint32_t hi = (j & 1) ? o4[2] : o4[0], lw = (j & 1) ? o4[3] : o4[1];
            const uint64_t U = ((uint64_t)hi << 21) | (lw >> 11);
            double o;
            RotVarU53::split(U, (uint32_t)nb, b, o);
            const double2 ev = RotVarU53::make(X[b], X[b + 1], a.shift[j], a.scale[j]);
            ent.x = (T)ev.x; ent.y = (T)ev.y;
            u = (T)fma(ev.y, o, ev.x);
            x_var = fma(X[b + 1] - X[b], o * 1.1102230246251565e-16, X[b]);
            word_var = hi;
        } else if (sizeof(T) == 8 && a.variant == kVarQ32) {   // C4': the fp32 pair (X~_b, Delta~_b)
            const float2 q = RotVarQ32::make(X[b], X[b + 1]);
            const double r = fma((double)lo, 2.3283064365386963e-10, 1.1641532182693481e-10);
            x_var = fma((double)q.y, r, (double)q.x);
            ent.x = (T)q.x; ent.y = (T)q.y;
            u = (T)((x_var - a.shift[j]) * a.scale[j]);
        } else if (sizeof(T) == 8 && a.word_map) {                   // the fast path's own split and map for this shape
            using SW = RotSplit<double, true>;
            uint32_t bw;
            double o;
            SW::split(word, (uint32_t)nb, (double)nb * 2.3283064365386963e-10, bw, o);
            b = bw;
            const double2 ew = SW::make(X[b], X[b + 1], a.shift[j], a.scale[j], (int)b, nb);
            ent.x = (T)ew.x; ent.y = (T)ew.y;
            u = (T)SW::u(ew, o);
        } else {
            ent = E::make(X[b], X[b + 1], a.shift[j], a.scale[j]);
            u = E::u(ent, lo);
        }
        jac[j & (NCH - 1)] *= ent.y;
        f.dim(u, FID == VEGAS_F_BW_POLY ? (j >> 2) : 0, j & 3, ctx);
        a.words[(size_t)q * dim + j] = word_var;
        a.bins[(size_t)q * dim + j] = (int32_t)b;
        a.x[(size_t)q * dim + j] = (sizeof(T) == 8 && a.variant != 0) ? x_var
                                   : (sizeof(T) == 8) ? fma(X[b + 1] - X[b], offset_f64(lo), X[b])
                                                     : (double)fmaf((float)(X[b + 1] - X[b]),
                                                                    offset_f32_scaled(lo, 5.9604644775390625e-08f, 2.98023223876953125e-08f),
                                                                    (float)X[b]);
    }
    a.fJ[q] = (double)f.value(jac, (T)a.fin0, (T)a.fin1) * a.post_scale;
}

// =============================================================================================
// Launchers
// =============================================================================================
template <int FID, typename T, int NBLK>
static cudaError_t launch_iterate_t(const IterArgs& a, const FParams<T>& fp, int blocks, int threads,
                                    size_t shmem, cudaStream_t st) {
    auto kern = k_iterate<FID, T, NBLK>;
    static size_t configured_dev[kMaxDevices] = {};   // per instantiation and device: the attribute is per context
    int dev_ = 0;
    if (cudaGetDevice(&dev_) != cudaSuccess || dev_ < 0 || dev_ >= kMaxDevices) return cudaErrorInvalidDevice;
    {
        // grids on different host threads may launch the same kernel: the cache and the attribute change together
        static std::mutex configured_mutex;
        std::lock_guard<std::mutex> lock(configured_mutex);
        size_t& configured = configured_dev[dev_];
        if (shmem > configured) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmem);
            if (e != cudaSuccess) return e;
            configured = shmem;
        }
    }
    kern<<<blocks, threads, shmem, st>>>(a, fp);
    return cudaGetLastError();
}

template <int FID, typename T>
static cudaError_t launch_iterate_nblk(const IterArgs& a, const FParams<T>& fp, int blocks, int threads,
                                       size_t shmem, cudaStream_t st) {
    switch ((a.dim + 3) / 4) {
    case 1: return launch_iterate_t<FID, T, 1>(a, fp, blocks, threads, shmem, st);
    case 2: return launch_iterate_t<FID, T, 2>(a, fp, blocks, threads, shmem, st);
    case 3: return launch_iterate_t<FID, T, 3>(a, fp, blocks, threads, shmem, st);
    case 4: return launch_iterate_t<FID, T, 4>(a, fp, blocks, threads, shmem, st);
    case 5: return launch_iterate_t<FID, T, 5>(a, fp, blocks, threads, shmem, st);
    case 6: return launch_iterate_t<FID, T, 6>(a, fp, blocks, threads, shmem, st);
    case 7: return launch_iterate_t<FID, T, 7>(a, fp, blocks, threads, shmem, st);
    case 8: return launch_iterate_t<FID, T, 8>(a, fp, blocks, threads, shmem, st);
    default: return cudaErrorInvalidValue;
    }
}

template <typename T>
static cudaError_t launch_iterate_fid(int fid, const IterArgs& a, const FParams<T>& fp, int blocks,
                                      int threads, size_t shmem, cudaStream_t st) {
    switch (fid) {
    case VEGAS_F_CONST: return launch_iterate_nblk<VEGAS_F_CONST, T>(a, fp, blocks, threads, shmem, st);
    case VEGAS_F_GAUSS: return launch_iterate_nblk<VEGAS_F_GAUSS, T>(a, fp, blocks, threads, shmem, st);
    case VEGAS_F_GENZ_PRODUCT_PEAK:
        return launch_iterate_nblk<VEGAS_F_GENZ_PRODUCT_PEAK, T>(a, fp, blocks, threads, shmem, st);
    case VEGAS_F_BW_POLY: return launch_iterate_nblk<VEGAS_F_BW_POLY, T>(a, fp, blocks, threads, shmem, st);
    case VEGAS_F_GENZ_DISCONTINUOUS:
        return launch_iterate_nblk<VEGAS_F_GENZ_DISCONTINUOUS, T>(a, fp, blocks, threads, shmem, st);
    default: return cudaErrorInvalidValue;
    }
}

template <typename T>
static void convert_params(const double* src, FParams<T>& dst) {
    for (int i = 0; i < VEGAS_MAX_PARAMS; ++i) dst.p[i] = (T)src[i];
}

cudaError_t launch_iterate(int fid, int precision, const IterArgs& a, const double* derived_params,
                           int blocks, int threads, size_t shmem, cudaStream_t st) {
    if (precision == VEGAS_FP64) {
        FParams<double> fp;
        convert_params(derived_params, fp);
        return launch_iterate_fid<double>(fid, a, fp, blocks, threads, shmem, st);
    }
    FParams<float> fp;
    convert_params(derived_params, fp);
    return launch_iterate_fid<float>(fid, a, fp, blocks, threads, shmem, st);
}

size_t iterate_shared_bytes(int dim, int n_bins, int precision, int table_copies, int hist_copies) {
    const size_t nent = (size_t)dim * n_bins;
    const size_t entry = precision == VEGAS_FP64 ? 16 : 8;
    return entry * nent * table_copies + 8 * nent * hist_copies + 2 * sizeof(dd) * (kIterMaxThreads / 32);
}

cudaError_t launch_reduce(const double* partials, int n_parts, int n_tot, double* totals, cudaStream_t st) {
    const int threads = 256;                                  // k_reduce: 8 warps = 8 slices of the CTA partials
    // ordinary launch: launched early, its CTAs would sit beside the fused kernel's on SMs with shared memory to spare
    k_reduce<<<1 + (n_tot - 4 + 31) / 32, threads, 0, st>>>(partials, n_parts, n_tot, totals);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const double* totals, double n_events, double* result, cudaStream_t st) {
    return launch_pdl(k_finalize, dim3(1), dim3(32), 0, st, totals, n_events, result);
}

cudaError_t launch_refine(double* edges, const double* hist, int dim, int n_bins, double alpha, int* status,
                          cudaStream_t st) {
    const int threads = ((n_bins + 31) / 32) * 32;
    return launch_pdl(k_refine, dim3(dim), dim3(threads), 0, st, edges, hist, n_bins, alpha, status);
}

template <typename T>
static cudaError_t launch_debug_t(int fid, const DebugArgs& a, const FParams<T>& fp, cudaStream_t st) {
    const int threads = 128;
    const int blocks = (int)((a.count + threads - 1) / threads);
    switch (fid) {
    case VEGAS_F_CONST: k_debug<VEGAS_F_CONST, T><<<blocks, threads, 0, st>>>(a, fp); break;
    case VEGAS_F_GAUSS: k_debug<VEGAS_F_GAUSS, T><<<blocks, threads, 0, st>>>(a, fp); break;
    case VEGAS_F_GENZ_PRODUCT_PEAK: k_debug<VEGAS_F_GENZ_PRODUCT_PEAK, T><<<blocks, threads, 0, st>>>(a, fp); break;
    case VEGAS_F_BW_POLY: k_debug<VEGAS_F_BW_POLY, T><<<blocks, threads, 0, st>>>(a, fp); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

template <typename T>
static cudaError_t launch_debug_rot_t(int fid, const DebugArgs& a, cudaStream_t st) {
    const int threads = 128;
    const int blocks = (int)((a.count + threads - 1) / threads);
    switch (fid) {
    case VEGAS_F_CONST: k_debug_rot<VEGAS_F_CONST, T><<<blocks, threads, 0, st>>>(a); break;
    case VEGAS_F_GAUSS: k_debug_rot<VEGAS_F_GAUSS, T><<<blocks, threads, 0, st>>>(a); break;
    case VEGAS_F_GENZ_PRODUCT_PEAK: k_debug_rot<VEGAS_F_GENZ_PRODUCT_PEAK, T><<<blocks, threads, 0, st>>>(a); break;
    case VEGAS_F_BW_POLY: k_debug_rot<VEGAS_F_BW_POLY, T><<<blocks, threads, 0, st>>>(a); break;
    case VEGAS_F_GENZ_DISCONTINUOUS: k_debug_rot<VEGAS_F_GENZ_DISCONTINUOUS, T><<<blocks, threads, 0, st>>>(a); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_accumulate_batch(const double* f, const double* J, const int32_t* bins, uint32_t count, int dim,
                                    int n_bins, double* partials, int blocks, cudaStream_t st) {
    const size_t shmem = sizeof(double) * (size_t)dim * n_bins + 2 * sizeof(dd) * 8;
    static size_t configured_dev[kMaxDevices] = {};   // per device: the attribute is per context
    int dev_ = 0;
    if (cudaGetDevice(&dev_) != cudaSuccess || dev_ < 0 || dev_ >= kMaxDevices) return cudaErrorInvalidDevice;
    {
        // grids on different host threads may launch the same kernel: the cache and the attribute change together
        static std::mutex configured_mutex;
        std::lock_guard<std::mutex> lock(configured_mutex);
        size_t& configured = configured_dev[dev_];
        if (shmem > configured) {
            cudaError_t e = cudaFuncSetAttribute(k_accumulate_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmem);
            if (e != cudaSuccess) return e;
            configured = shmem;
        }
    }
    k_accumulate_batch<<<blocks, 256, shmem, st>>>(f, J, bins, count, dim, n_bins, partials);
    return cudaGetLastError();
}

cudaError_t launch_debug(int fid, int precision, bool rot_path, const DebugArgs& a, const double* derived_params,
                         cudaStream_t st) {
    if (rot_path)
        return precision == VEGAS_FP64 ? launch_debug_rot_t<double>(fid, a, st) : launch_debug_rot_t<float>(fid, a, st);
    if (precision == VEGAS_FP64) {
        FParams<double> fp;
        convert_params(derived_params, fp);
        return launch_debug_t<double>(fid, a, fp, st);
    }
    FParams<float> fp;
    convert_params(derived_params, fp);
    return launch_debug_t<float>(fid, a, fp, st);
}

}  // namespace vegas
