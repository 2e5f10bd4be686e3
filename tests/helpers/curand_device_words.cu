// Test helper (GPU box only): cuRAND's own DEVICE generator, as a library cross-check of the counter/key layout C2
// ("On the box: equality with cuRAND's device curand4 under the mapping in C2"; PAPER.md:49-51 leaves
// "how to generate the random numbers" open).  For every input line "seed e iteration block" (hex, 64/64/32/32 bits)
// one thread runs
//     curand_init(seed, /*subsequence*/ e, /*offset*/ 4 * ((uint64)iteration << 32 | block), &st);  curand4(&st);
// and the program prints the four 32-bit outputs (hex).  C2 says these are the Philox words of dimensions
// 4*block .. 4*block+3 of event e of that iteration.  Nothing of the library or of the oracle is included here.
#include <cuda_runtime.h>
#include <curand_kernel.h>

#include <cstdio>
#include <vector>

struct Query { unsigned long long seed, e; unsigned int iteration, block; };

__global__ void k_curand4(const Query* q, uint4* out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    curandStatePhilox4_32_10_t st;
    curand_init(q[i].seed, q[i].e, 4ull * (((unsigned long long)q[i].iteration << 32) | q[i].block), &st);
    out[i] = curand4(&st);
}

int main() {
    std::vector<Query> qs;
    Query q;
    while (scanf("%llx %llx %x %x", &q.seed, &q.e, &q.iteration, &q.block) == 4) qs.push_back(q);
    const int n = (int)qs.size();
    if (n == 0) return 0;
    Query* dq = nullptr;
    uint4* dout = nullptr;
    if (cudaMalloc(&dq, n * sizeof(Query)) != cudaSuccess || cudaMalloc(&dout, n * sizeof(uint4)) != cudaSuccess) return 2;
    cudaMemcpy(dq, qs.data(), n * sizeof(Query), cudaMemcpyHostToDevice);
    k_curand4<<<(n + 127) / 128, 128>>>(dq, dout, n);
    std::vector<uint4> out(n);
    if (cudaMemcpy(out.data(), dout, n * sizeof(uint4), cudaMemcpyDeviceToHost) != cudaSuccess) return 3;
    for (const uint4& o : out) printf("%08x %08x %08x %08x\n", o.x, o.y, o.z, o.w);
    cudaFree(dq);
    cudaFree(dout);
    return 0;
}
