// vegas_rot_inst.cu -- instantiates k_iterate_rot<ROT_FID, T, DIM, ROT_VAR> for DIM = 1..32 (BW_POLY: 2..32).
// Compiled once per (ROT_FID, ROT_FP, ROT_VAR) triple by build.py so that they build in parallel
// (ROT_VAR: 0 = the method, 1 = 53-bit uniforms, 2 = fp32-rounded table; the variants are fp64 only).
#include "vegas_iterate_rot.cuh"

#include <mutex>

#ifndef ROT_FID
#error "compile with -DROT_FID=<integrand id> -DROT_FP=<64|32>"
#endif

#ifndef ROT_VAR
#define ROT_VAR 0
#endif

namespace vegas {

#if ROT_FP == 64
using RT = double;
#else
using RT = float;
#endif

template <int DIM, bool PAIR>
static cudaError_t go_kernel(const RotArgs& a, int blocks, int threads, size_t shmem, cudaStream_t st) {
    auto kern = k_iterate_rot<ROT_FID, RT, DIM, ROT_VAR, PAIR>;
    static size_t configured_dev[kMaxDevices] = {};   // per kernel and device: the attribute is per context
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
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(blocks);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = shmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = a.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, a);
}

// rings of the 3-block shapes run the two-events-per-hold kernel (rot_pair_hold)
template <int DIM>
static cudaError_t go(const RotArgs& a, int blocks, int threads, size_t shmem, cudaStream_t st) {
    if constexpr (rot_pair_hold(ROT_FID, DIM, ROT_VAR)) {
        if (a.ring > 1) return go_kernel<DIM, true>(a, blocks, threads, shmem, st);
    }
    return go_kernel<DIM, false>(a, blocks, threads, shmem, st);
}

template <>
cudaError_t launch_iterate_rot<ROT_FID, RT, ROT_VAR>(int dim, const RotArgs& a, int blocks, int threads, size_t shmem,
                                            cudaStream_t st) {
    switch (dim) {
#define CASE(D) case D: return go<D>(a, blocks, threads, shmem, st);
#if ROT_FID != VEGAS_F_BW_POLY
        CASE(1)
#endif
        CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
        CASE(9) CASE(10) CASE(11) CASE(12) CASE(13) CASE(14) CASE(15) CASE(16)
        CASE(17) CASE(18) CASE(19) CASE(20) CASE(21) CASE(22) CASE(23) CASE(24)
        CASE(25) CASE(26) CASE(27) CASE(28) CASE(29) CASE(30) CASE(31) CASE(32)
#undef CASE
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace vegas
