// common.cuh -- shared device/host declarations of librosen (product path; never includes oracle/).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "philox.cuh"

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
    PhiloxKeys rk;              // its ten round keys
    double     ln_shift;        // L
    DevOutputs out;
    Partial*   partials;        // [n_vblocks]
    uint32_t   chunk;           // chains per virtual block (multiple of 256)
    uint32_t   n_vblocks;       // ceil(n_chains / chunk) <= kMaxPartials
    uint32_t*  vb_counter;      // zeroed before the launch: blocks draw virtual blocks from it (load balance only;
                                // partials[v] never depends on which block computed it)
};

struct ChainRecord;
struct RealParams {
    int32_t    N;
    int32_t    k;
    uint64_t   n_chains;
    uint64_t   chain_offset;
    uint32_t   key0, key1;      // (round keys as parameters, as in LatticeParams, measured slower here: 25.3 -> 25.9 ms at config 3)
    float      b, sigma2, prefilter2;   // bond length, sigma^2 (fp32), conservative candidate radius^2
    double     ln_shift;
    DevOutputs out;
    Partial*   partials;        // [n_vblocks]
    uint32_t   chunk;           // chains per virtual block (multiple of 256)
    uint32_t   n_vblocks;
    uint32_t*  vb_counter;      // as in LatticeParams
    uint32_t*  done;            // null, or [n_vblocks] flags in mapped host memory: set when a virtual block's outputs are stored
                                // (the host streams finished conformations out while the kernel runs: DESIGN.md 5.4)
    // square-well model (rosen_realspace_generate_model): rec != nullptr selects the WELL kernels
    float        well2;         // fl32(fl32(lambda sigma)^2)
    ChainRecord* rec;           // [n_chains]: per-chain records instead of block partials (shift = largest lnW of the call)
    uint64_t     Q[32];         // fixed-point Boltzmann factors round(q^c 2^16)
};

// Long-chain lattice path (lattice_hash.cu): one fixed-size record per chain, reduced afterwards in a fixed order.
struct ChainRecord {
    double   lnW, ree2, rg2;    // -inf / 0 / 0 for a dead chain
    uint32_t steps, alive;      // attempted steps; 1 = reached N monomers
    uint64_t digest;
};

struct HashParams {
    int32_t    N;
    uint64_t   n_chains;
    uint64_t   chain_offset;
    uint32_t   key0, key1;
    double     ln_shift;
    DevOutputs out;
    Partial*   partials;        // [n_vblocks]
    uint32_t   chunk;           // chains per virtual block (multiple of 256)
    uint32_t   n_vblocks;
    ChainRecord* rec;           // [n_chains]
    uint64_t*  tables;          // [launched threads][entries] 16-byte entries, zeroed before the launch
    uint32_t   entries;         // entries per chain table (even, >= N + 1)
    unsigned long long* ticket; // zeroed before the launch: lanes draw chain indices from it (load balance only)
    double*    lmax;            // [kMaxPartials + 1] scratch, or null: N <= 512, fixed shift ln_shift (reading A18)
    uint32_t*  gen_store;       // [launched threads] each thread's generation counter, kept across calls of one table layout
};

// Lattice model path (lattice_model.cu): z = 6 / 26 trial set, contact energy, records + dynamic shift.
struct ModelParams {
    int32_t    N;
    int32_t    z;
    uint64_t   n_chains;
    uint64_t   chain_offset;
    uint32_t   key0, key1;
    uint64_t   Q[32];           // fixed-point Boltzmann factors round(q^c 2^16)
    DevOutputs out;
    Partial*   partials;        // [n_vblocks]
    uint32_t   chunk;
    uint32_t   n_vblocks;
    ChainRecord* rec;           // [n_chains]
    double*    lmax;            // [kMaxPartials + 1] scratch of the max pass
};

// PERM (lattice_perm.cu): one record per tour, thresholds in device memory.
struct PermParams {
    int32_t    N;
    uint64_t   n_tours;
    uint64_t   tour_offset;
    uint32_t   key0, key1;
    const double* ln_lo;        // [N + 1] device copies of the caller's thresholds (index = number of monomers)
    const double* ln_hi;
    double     ln_ref;          // reference of the leaf weights inside a tour: w = exp(lnW - ln_ref)
    uint32_t   max_nodes;
    DevOutputs out;
    Partial*   partials;
    uint32_t   chunk;
    uint32_t   n_vblocks;
    ChainRecord* rec;           // [n_tours]; alive bit 0 = the tour has a leaf, bit 1 = stopped at max_nodes
    double*    lmax;
    unsigned long long* ticket; // zeroed before the launch
};

constexpr uint32_t kRealLongCandCap = 160;

// Long-chain real-space path (realspace_long.cu): one warp grows one chain; chain, cell table and cell lists in HBM.
struct RealLongParams {
    int32_t    N;
    int32_t    k;
    uint64_t   n_chains;
    uint64_t   chain_offset;
    uint32_t   key0, key1;
    float      b, sigma2, prefilter2;   // as RealParams
    float      inv_cell;        // 1 / cell edge; cell edge >= candidate radius x (1 + 2^-6)
    double     ln_shift;
    DevOutputs out;
    Partial*   partials;        // [n_vblocks]
    uint32_t   chunk;           // chains per virtual block (multiple of 256)
    uint32_t   n_vblocks;
    ChainRecord* rec;           // [n_chains]
    unsigned char* work;        // [launched warps][warp_bytes], zeroed before the launch
    uint64_t   warp_bytes;      // float4 r[n_pad] (x, y, z, list link) | 16-byte cell entries [entries], padded to 256
    uint32_t   n_pad;           // N rounded up to 8
    uint32_t   cand_cap;        // candidates buffered per warp before a flush: 33 .. kRealLongCandCap
    uint32_t   entries;         // cell-table entries per chain (even, >= N + 1)
    unsigned long long* ticket; // zeroed before the launch: warps draw chain indices from it (load balance only)
    double*    lmax;            // [kMaxPartials + 1] scratch, or null: N <= 2048, fixed shift ln_shift (reading A18)
    uint32_t*  gen_store;       // [launched warps] each warp's generation counter, kept across calls of one workspace layout
};

// The ensemble reduction is tied to VIRTUAL blocks, not to the launch grid: virtual block v owns the
// chain range [v*chunk, (v+1)*chunk) and produces partials[v] with a fixed thread mapping and tree, so
// the sums depend on (n_chains, N) only -- never on the grid size, occupancy, output variant or GPU.
// (Real space: chunk >= 256 because one chain occupies a lane group for ~100x longer than a lattice chain.)
constexpr int kMaxPartials = 8192;
constexpr uint32_t kMinChunk = 2048;

// chunk = chains per virtual block: >= kMinChunk, a multiple of 256, and large enough for <= kMaxPartials blocks.
inline void partition_chains(uint64_t n_chains, uint32_t* chunk, uint32_t* n_vblocks, uint32_t min_chunk = kMinChunk)
{
    uint64_t c = (n_chains + kMaxPartials - 1) / kMaxPartials;
    c = (c + 255) / 256 * 256;
    if (c < min_chunk) c = min_chunk;
    *chunk = (uint32_t)c;
    *n_vblocks = (uint32_t)((n_chains + c - 1) / c);
}

// launchers (lattice.cu / realspace.cu / reduce.cu). Return the number of kernels launched or
// a negative ROSEN_E* code; *kernel_name receives a static string naming the variant chosen.
int launch_lattice(const LatticeParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out);
// lattice_hash.cu: table geometry for chain length N, resident thread capacity of the device, launch (generation
// kernel over n_threads = multiple of 256 threads, then the per-record first reduction pass).
uint32_t hash_entries(int32_t N);
int hash_max_threads(int* threads_out, int blocks_per_sm_cap);   // cap: 0 = none (tuning knob; results do not depend on it)
uint32_t lattice_hash_gen_max();  // largest generation tag of a table entry (the counter wraps beyond it)
int launch_lattice_hash(const HashParams& p, int n_threads, cudaStream_t stream, const char** kernel_name);
// reduce_records_kernel of lattice_hash.cu: first reduction pass over per-chain records (+ optional per-chain outputs)
// lmax != nullptr: first find L = max lnW (two launches), left in lmax[kMaxPartials]. Returns the launches made.
int launch_reduce_records(const ChainRecord* rec, uint64_t n_chains, uint32_t chunk, uint32_t n_vblocks, double ln_shift,
                          double* lmax, const DevOutputs& out, Partial* partials, cudaStream_t stream);
// realspace_long.cu: resident warp capacity, launch over n_warps (multiple of 8) warps + the record reduction
int real_long_max_warps(int k, int* warps_out);
uint32_t real_long_gen_max();
int launch_realspace_long(const RealLongParams& p, int n_warps, cudaStream_t stream, const char** kernel_name);
int launch_realspace(const RealParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out);
// realspace.cu: the D1 store phase alone over a resident synthetic chain (measurement entry rosen_realspace_dump_probe)
int launch_dump_probe(int N, uint64_t n_chains, float* conf, double* lnW, cudaStream_t stream);
// lattice_model.cu: generation kernel + record reduction (max pass included); returns the launches made
int launch_lattice_model(const ModelParams& p, cudaStream_t stream, const char** kernel_name);
// lattice_perm.cu: tour kernel + record reduction; returns the launches made
int launch_lattice_perm(const PermParams& p, cudaStream_t stream, const char** kernel_name);
// realspace.cu: the direction map of DESIGN.md 3.3 alone, out[3 i ..] = direction(wz[i], wphi[i]) (device pointers)
int launch_direction_eval(const uint32_t* wz, const uint32_t* wphi, uint64_t n, float* out, cudaStream_t stream);
int launch_finalize(const Partial* partials, int n_partials, uint64_t n_chains, double ln_shift, const double* ln_shift_dev,
                    void* summary_dev, cudaStream_t stream);   // summary_dev: rosen_summary* in device memory

}  // namespace rosen
