// vegas_kernels.h -- host-visible launchers of the sm_100a kernels (vegas_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/vegas.h"

namespace vegas {

#ifndef VEGAS_ITER_MAX_THREADS
#define VEGAS_ITER_MAX_THREADS 512
#endif
#ifndef VEGAS_ITER_MIN_BLOCKS
#define VEGAS_ITER_MIN_BLOCKS 1
#endif
constexpr int kMaxDevices = 64;                          // per-device launch-attribute caches
constexpr int kIterMaxThreads = VEGAS_ITER_MAX_THREADS;   // __launch_bounds__ of K1
constexpr int kIterMinBlocks = VEGAS_ITER_MIN_BLOCKS;

struct IterArgs {
    const double* edges;            // device, [dim][n_bins+1] master grid
    double* partials;               // device, [blocks][4 + dim*n_bins]
    unsigned long long first_event; // global index of the first event of this launch (C2)
    unsigned long long count;       // events in this launch
    uint32_t key0, key1;            // seed lo, seed hi
    uint32_t iteration;
    int dim, n_bins;
    int log_ct, log_ch;             // log2 of the table / histogram copy counts
    double jac_scale;               // BW_POLY: fp64: n_bins^dim (the table holds Delta); fp32: 1
    // CONST, GAUSS, GENZ: the affine map and constants of the fast path (vegas_iterate_rot.cuh: RotEntry, IntegrandU),
    // so that both kernels form u_j, f and v by the same arithmetic (C11: same fp32 accuracy and range)
    double post_scale, fin0, fin1, jac_init;
    double shift[VEGAS_MAX_DIM], scale[VEGAS_MAX_DIM];
};

struct DebugArgs {
    const double* edges;
    unsigned long long first_event;
    uint32_t count;
    uint32_t key0, key1, iteration;
    int dim, n_bins;
    double jac_scale;
    uint32_t* words;
    int32_t* bins;
    double* x;
    double* fJ;
    // fast ("rotated") path only: the affine map and constants of vegas_iterate_rot.cuh
    double post_scale, fin0, fin1, jac_init;
    double shift[VEGAS_MAX_DIM], scale[VEGAS_MAX_DIM];
    double fpar[5 * VEGAS_MAX_DIM]; // RotArgs::fpar (kRotParams)
    int variant;                    // VEGAS_VARIANT_* (fp64 fast path only): the sampling map of this grid
    int word_map;                   // fp64: this shape's fast-path kernel uses the word-affine table entries (rot_word_map)
};

size_t iterate_shared_bytes(int dim, int n_bins, int precision, int table_copies, int hist_copies);

cudaError_t launch_iterate(int fid, int precision, const IterArgs& a, const double* derived_params,
                           int blocks, int threads, size_t shmem, cudaStream_t st);
cudaError_t launch_reduce(const double* partials, int n_parts, int n_tot, double* totals, cudaStream_t st);
cudaError_t launch_finalize(const double* totals, double n_events, double* result, cudaStream_t st);
cudaError_t launch_refine(double* edges, const double* hist, int dim, int n_bins, double alpha, int* status,
                          cudaStream_t st);
cudaError_t launch_accumulate_batch(const double* f, const double* J, const int32_t* bins, uint32_t count, int dim,
                                    int n_bins, double* partials, int blocks, cudaStream_t st);
cudaError_t launch_debug(int fid, int precision, bool rot_path, const DebugArgs& a, const double* derived_params,
                         cudaStream_t st);

}  // namespace vegas
