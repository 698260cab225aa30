// reduce.cuh -- deterministic ensemble reduction (E1): warp shuffle tree -> block tree ->
// block partial; reduce.cu sums the block partials in a second kernel. No atomics anywhere, so
// the result depends only on the (fixed) launch geometry, never on scheduling.
#pragma once
#include "common.cuh"

namespace rosen {

__device__ __forceinline__ double shfl_down_f64(double v, int delta)
{
    return __shfl_down_sync(0xffffffffu, v, delta);
}
__device__ __forceinline__ uint64_t shfl_down_u64(uint64_t v, int delta)
{
    return __shfl_down_sync(0xffffffffu, (unsigned long long)v, delta);
}

__device__ __forceinline__ Partial partial_zero()
{
    Partial z; z.sum_w = z.sum_w_ree2 = z.sum_w_rg2 = z.sum_w2 = 0.0;
    z.n_dead = z.n_steps = z.digest_xor = z.digest_sum = 0; return z;
}

__device__ __forceinline__ void partial_combine(Partial& a, const Partial& b)
{
    a.sum_w += b.sum_w; a.sum_w_ree2 += b.sum_w_ree2; a.sum_w_rg2 += b.sum_w_rg2; a.sum_w2 += b.sum_w2;
    a.n_dead += b.n_dead; a.n_steps += b.n_steps; a.digest_xor ^= b.digest_xor; a.digest_sum += b.digest_sum;
}

__device__ __forceinline__ Partial warp_reduce(Partial v)
{
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
        Partial o;
        o.sum_w = shfl_down_f64(v.sum_w, d); o.sum_w_ree2 = shfl_down_f64(v.sum_w_ree2, d);
        o.sum_w_rg2 = shfl_down_f64(v.sum_w_rg2, d); o.sum_w2 = shfl_down_f64(v.sum_w2, d);
        o.n_dead = shfl_down_u64(v.n_dead, d); o.n_steps = shfl_down_u64(v.n_steps, d);
        o.digest_xor = shfl_down_u64(v.digest_xor, d); o.digest_sum = shfl_down_u64(v.digest_sum, d);
        partial_combine(v, o);
    }
    return v;   // lane 0 holds the warp total (fixed tree)
}

// All threads of the block call this (after their last use of `scratch`); thread 0 writes the
// block partial. scratch: >= (blockDim.x/32) Partials of shared memory.
__device__ __forceinline__ void block_reduce_store(Partial v, Partial* scratch, Partial* dst)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    v = warp_reduce(v);
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        Partial t = scratch[0];
        for (int w = 1; w < nwarp; ++w) partial_combine(t, scratch[w]);   // warp order
        *dst = t;
    }
}

}  // namespace rosen
