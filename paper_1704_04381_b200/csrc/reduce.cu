// reduce.cu -- second pass of the two-pass fp64 ensemble reduction (BASELINE config 2:
// "deterministic two-pass fp64 reduction"): one block sums the per-block partials in a fixed order
// and writes the finished rosen_summary (sums + derived fields, Eq. 2, Eq. 6 :362).
#include "../../include/rosen.h"
#include "reduce.cuh"

namespace rosen {

__global__ void __launch_bounds__(256) finalize_kernel(const Partial* __restrict__ partials, int n,
                                                       uint64_t n_chains, double ln_shift, const double* ln_shift_dev,
                                                       rosen_summary* out)
{
    if (ln_shift_dev) ln_shift = *ln_shift_dev;        // long chains: L = max lnW, found on the device (reading A18)
    __shared__ Partial scratch[8];
    __shared__ Partial total;
    Partial acc = partial_zero();
    for (int i = threadIdx.x; i < n; i += 256) partial_combine(acc, partials[i]);   // strided, fixed order
    block_reduce_store(acc, scratch, &total);
    if (threadIdx.x == 0) {
        const Partial t = total;
        rosen_summary s;
        s.n_chains = n_chains; s.n_dead = t.n_dead; s.n_steps_attempted = t.n_steps; s.ln_shift = ln_shift;
        s.sum_w = t.sum_w; s.sum_w_ree2 = t.sum_w_ree2; s.sum_w_rg2 = t.sum_w_rg2; s.sum_w2 = t.sum_w2;
        s.mean_ree2 = t.sum_w_ree2 / t.sum_w;
        s.mean_rg2 = t.sum_w_rg2 / t.sum_w;
        s.attrition = (double)t.n_dead / (double)n_chains;
        s.ln_mean_W = ln_shift + log(t.sum_w / (double)n_chains);
        s.digest_xor = t.digest_xor; s.digest_sum = t.digest_sum;
        *out = s;
    }
}

int launch_finalize(const Partial* partials, int n_partials, uint64_t n_chains, double ln_shift, const double* ln_shift_dev,
                    void* summary_dev, cudaStream_t stream)
{
    finalize_kernel<<<1, 256, 0, stream>>>(partials, n_partials, n_chains, ln_shift, ln_shift_dev,
                                           static_cast<rosen_summary*>(summary_dev));
    return cudaGetLastError() == cudaSuccess ? 1 : -3;
}

}  // namespace rosen
