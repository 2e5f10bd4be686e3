// vegas_user.h -- run-time compiled user integrands (vegas_user.cu): host-side interface used by vegas_api.cu.
#pragma once
#include <cuda_runtime.h>

#include <string>

#include "vegas_iterate_rot.cuh"

namespace vegas {

struct UserKernel {
    cudaLibrary_t library = nullptr;   // loaded cubin (owned; user_unload releases it)
    cudaKernel_t kernel = nullptr;     // k_iterate_rot<VEGAS_F_USER, double, dim>
    cudaKernel_t kernel32 = nullptr;   // k_iterate_rot<VEGAS_F_USER, float, dim>: the fp32 sampling map (C11) around the same f
    size_t smem_configured = 0, smem_configured32 = 0;
    int dim = 0;
};

// Compile `user_source` (defines struct vegas_user_integrand, see include/vegas.h) for `dim` dimensions.
// Returns 0, -1 (the source does not compile: *log holds the compiler output) or -2 (NVRTC / runtime failure:
// *err says which).  On success *out replaces whatever it held before.
int user_compile(const char* user_source, int dim, std::string* log, UserKernel* out, std::string* err);
cudaError_t user_launch(UserKernel* uk, bool fp32, const RotArgs& a, int blocks, int threads, size_t shmem, cudaStream_t st);
void user_unload(UserKernel* uk);

}  // namespace vegas
