// reduce.cu -- second pass of the two-pass fp64 ensemble reduction (BASELINE config 2:
// "deterministic two-pass fp64 reduction"): one block sums the per-block partials in a fixed order.
#include "reduce.cuh"

namespace rosen {

__global__ void __launch_bounds__(256) finalize_kernel(const Partial* __restrict__ partials, int n, Partial* total)
{
    __shared__ Partial scratch[8];
    Partial acc = partial_zero();
    for (int i = threadIdx.x; i < n; i += 256) partial_combine(acc, partials[i]);   // strided, fixed order
    block_reduce_store(acc, scratch, total);
}

int launch_finalize(const Partial* partials, int n_partials, Partial* total, cudaStream_t stream)
{
    finalize_kernel<<<1, 256, 0, stream>>>(partials, n_partials, total);
    return cudaGetLastError() == cudaSuccess ? 1 : -3;
}

}  // namespace rosen
