// common.cuh -- shared device/host declarations of librosen (product path; never includes oracle/).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rosen {

// Per-block partial of the ensemble sums (E1; Eq. 2).
struct Partial {
    double   sum_w, sum_w_ree2, sum_w_rg2, sum_w2;
    uint64_t n_dead, n_steps, digest_xor, digest_sum;
};

// Device pointers of the optional per-chain outputs (all may be null).
struct DevOutputs {
    double*   lnW;
    uint8_t*  alive;
    uint8_t*  m_seq;
    uint64_t* digest;
    void*     conf;
    double*   ree2;
    double*   rg2;
};

struct LatticeParams {
    int32_t    N;
    uint64_t   n_chains;
    uint64_t   chain_offset;
    uint32_t   key0, key1;      // Philox key = seed
    double     ln_shift;        // L
    DevOutputs out;
    Partial*   partials;        // [gridDim.x]
};

struct RealParams {
    int32_t    N;
    int32_t    k;
    uint64_t   n_chains;
    uint64_t   chain_offset;
    uint32_t   key0, key1;
    float      b, sigma2, prefilter2;   // bond length, sigma^2 (fp32), conservative candidate radius^2
    double     ln_shift;
    DevOutputs out;
    Partial*   partials;
};

constexpr int kMaxPartials = 4096;   // upper bound on gridDim.x of the generation kernels

// launchers (lattice.cu / realspace.cu / reduce.cu). Return the number of kernels launched or
// a negative ROSEN_E* code; *kernel_name receives a static string naming the variant chosen.
int launch_lattice(const LatticeParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out);
int launch_realspace(const RealParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out);
int launch_finalize(const Partial* partials, int n_partials, uint64_t n_chains, double ln_shift,
                    void* summary_dev, cudaStream_t stream);   // summary_dev: rosen_summary* in device memory

}  // namespace rosen
