// lattice_model.cu -- lattice chains with other trial sets and Boltzmann-weighted trials (
// DESIGN.md 3.6, readings A19-A21): the z = 6 or z = 26 neighbourhood (sec. 3.3.2 "z = 26 possible lattice
// space") and a contact energy -eps per non-bonded neighbour pair (Eq. 1-2), i.e. Rosenbluth factors
// W_s = sum_t q^c_t over the free trials and a choice proportional to q^c_t, with fixed-point factors Q[c] = round(q^c 2^16).
//
// One thread grows one chain, 2 <= N <= 256. The chain is one packed 32-bit key per monomer (3 x 10-bit fields, bias 512)
// in shared memory, laid out [monomer][thread] so that the lock-step scan of a warp touches every bank once. Each step
// scans the earlier monomers j <= s-2 once and records those inside the 5 x 5 x 5 box around r_{s-1} in a 125-bit map
// held in registers; every trial site and all its neighbours lie inside that box, so "is the site free" and "how many
// contacts would it make" are a bit test and a popcount of the map under a precomputed neighbourhood mask.
// Results go to one record per chain; reduce_records_kernel (lattice_hash.cu) forms the deterministic sums with the
// largest lnW of the call as the shift (reading A18's mechanism).
#include <math_constants.h>
#include "common.cuh"
#include "philox.cuh"

namespace rosen {

namespace {

constexpr int kField = 10, kBias = 512;
constexpr uint32_t kFieldMask = (1u << kField) - 1u;

__device__ __forceinline__ uint64_t fold(uint64_t h, uint32_t m, uint32_t choice)
{
    return (h ^ (uint64_t)(m | (choice << 8))) * 0x100000001B3ull;
}

// trial d of the z-neighbourhood: z = 6: +x,-x,+y,-y,+z,-z; z = 26: rank of i = (dx+1) + 3(dy+1) + 9(dz+1), i != 13
template <int Z>
__device__ __forceinline__ void trial_offset(int d, int& ex, int& ey, int& ez)
{
    if (Z == 6) {
        const int a = d >> 1, sg = (d & 1) ? -1 : 1;
        ex = a == 0 ? sg : 0; ey = a == 1 ? sg : 0; ez = a == 2 ? sg : 0;
    } else {
        const int i = d < 13 ? d : d + 1;
        ex = i % 3 - 1; ey = (i / 3) % 3 - 1; ez = i / 9 - 1;
    }
}

template <int Z>
__device__ __forceinline__ bool neighbours(int dx, int dy, int dz)
{
    const int ax = abs(dx), ay = abs(dy), az = abs(dz);
    if (ax + ay + az == 0) return false;
    return Z == 6 ? ax + ay + az == 1 : (ax <= 1 && ay <= 1 && az <= 1);
}

// floor(u W / 2^32), W < 2^63
__device__ __forceinline__ uint64_t scaled_target(uint32_t u, uint64_t W)
{
    return (W >> 32) * (uint64_t)u + (((W & 0xFFFFFFFFull) * (uint64_t)u) >> 32);
}

// CONTACTS = false: every factor Q[c] is the same number (beta eps = 0: q = 1), so the contact counts cannot influence a
// weight or a choice and are not formed; the decisions are the same bits either way (the host picks the variant from Q).
template <int Z, bool TRAJ, bool CONTACTS>
__global__ void __launch_bounds__(256) lattice_model_kernel(const ModelParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t* Qs = reinterpret_cast<uint64_t*>(smem_raw);                    // [32] fixed-point factors
    uint64_t* nb = Qs + 32;                                                  // [Z][2] neighbourhood mask of trial site d in the box
    uint32_t* keys = reinterpret_cast<uint32_t*>(nb + 2 * Z);                // [N][blockDim.x]
    const int T = blockDim.x, tid = threadIdx.x, N = p.N;

    if (tid < 32) Qs[tid] = p.Q[tid];
    if (tid < Z) {
        int ex, ey, ez;
        trial_offset<Z>(tid, ex, ey, ez);
        uint64_t lo = 0, hi = 0;
        for (int idx = 0; idx < 125; ++idx) {
            const int x = idx % 5 - 2, y = (idx / 5) % 5 - 2, zc = idx / 25 - 2;
            if (neighbours<Z>(x - ex, y - ey, zc - ez)) { if (idx < 64) lo |= 1ull << idx; else hi |= 1ull << (idx - 64); }
        }
        nb[2 * tid] = lo; nb[2 * tid + 1] = hi;
    }
    __syncthreads();

    for (uint64_t idx = (uint64_t)blockIdx.x * T + tid; idx < p.n_chains; idx += (uint64_t)gridDim.x * T) {
        const uint64_t chain = p.chain_offset + idx;
        const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);
        int hx = 0, hy = 0, hz = 0;                                          // r_{s-1}
        int sx = 0, sy = 0, sz = 0, s2 = 0;
        double lnW = 0.0;
        uint32_t dead = 0;
        uint64_t dg = 0xCBF29CE484222325ull;
        uint32_t w4[4] = {0, 0, 0, 0};
        uint8_t* mrow = TRAJ && p.out.m_seq ? p.out.m_seq + idx * (uint64_t)(N - 1) : nullptr;
        int32_t* crow = TRAJ && p.out.conf ? reinterpret_cast<int32_t*>(p.out.conf) + idx * (uint64_t)N * 3 : nullptr;
        if (crow) { crow[0] = 0; crow[1] = 0; crow[2] = 0; }
        keys[tid] = (uint32_t)kBias | ((uint32_t)kBias << kField) | ((uint32_t)kBias << (2 * kField));

        int s = 1;
        for (; s < N; ++s) {
            if ((s & 3) == 0 || s == 1) philox4x32_10(c_lo, c_hi, (uint32_t)(s >> 2), 0u, p.key0, p.key1, w4);
            const uint32_t lo2 = (s & 1) ? w4[1] : w4[0], hi2 = (s & 1) ? w4[3] : w4[2];
            const uint32_t u = (s & 2) ? hi2 : lo2;

            // ---- occupancy of the 5 x 5 x 5 box around r_{s-1} by the monomers j <= s-2
            uint64_t mlo = 0, mhi = 0;
            const int bx = hx + kBias - 2, by = hy + kBias - 2, bz = hz + kBias - 2;
            for (int j = 0; j < s - 1; ++j) {
                const uint32_t key = keys[j * T + tid];
                const uint32_t ux = (key & kFieldMask) - (uint32_t)bx, uy = ((key >> kField) & kFieldMask) - (uint32_t)by,
                               uz = (key >> (2 * kField)) - (uint32_t)bz;
                if (ux < 5u && uy < 5u && uz < 5u) {
                    const uint32_t b = ux + 5u * uy + 25u * uz;
                    if (b < 64u) mlo |= 1ull << b; else mhi |= 1ull << (b - 64u);
                }
            }

            // ---- per trial: free?  contacts?  fixed-point factor
            uint64_t wq[Z];
            uint64_t W = 0;
            uint32_t m = 0;
#pragma unroll
            for (int d = 0; d < Z; ++d) {
                int ex, ey, ez;
                trial_offset<Z>(d, ex, ey, ez);
                const int site = 62 + ex + 5 * ey + 25 * ez;                 // compile-time after unrolling
                const bool occ = site < 64 ? ((mlo >> site) & 1ull) != 0ull : ((mhi >> (site - 64)) & 1ull) != 0ull;
                const int c = CONTACTS ? __popcll(mlo & nb[2 * d]) + __popcll(mhi & nb[2 * d + 1]) : 0;
                wq[d] = occ ? 0ull : Qs[c];
                W += wq[d]; m += occ ? 0u : 1u;
            }
            if (TRAJ && mrow) mrow[s - 1] = (uint8_t)m;
            if (m == 0u) { dead = (uint32_t)s; dg = fold(dg, 0u, 0xFFu); break; }
            lnW += log((double)W * 0x1p-16);

            // ---- the first trial whose cumulative sum exceeds floor(u W / 2^32)
            const uint64_t target = scaled_target(u, W);
            uint64_t cum = 0;
            int dsel = Z - 1;
            bool found = false;
#pragma unroll
            for (int d = 0; d < Z; ++d) {
                cum += wq[d];
                if (!found && cum > target) { found = true; dsel = d; }
            }
            int ex, ey, ez;
            trial_offset<Z>(dsel, ex, ey, ez);
            hx += ex; hy += ey; hz += ez;
            keys[s * T + tid] = (uint32_t)(hx + kBias) | ((uint32_t)(hy + kBias) << kField) | ((uint32_t)(hz + kBias) << (2 * kField));
            sx += hx; sy += hy; sz += hz; s2 += hx * hx + hy * hy + hz * hz;
            dg = fold(dg, m, (uint32_t)dsel);
            if (TRAJ && crow) { crow[3 * s] = hx; crow[3 * s + 1] = hy; crow[3 * s + 2] = hz; }
        }

        const bool alive = dead == 0u;
        if (TRAJ && !alive) {          // zero from the death step on (reading A13); m_seq[dead - 1] = 0 is already written
            if (crow) for (int q = (int)dead; q < N; ++q) { crow[3 * q] = 0; crow[3 * q + 1] = 0; crow[3 * q + 2] = 0; }
            if (mrow) for (int q = (int)dead; q < N - 1; ++q) mrow[q] = 0;
        }
        ChainRecord r;
        r.lnW = alive ? lnW : -CUDART_INF; r.ree2 = 0.0; r.rg2 = 0.0;
        if (alive) {
            r.ree2 = (double)(hx * hx + hy * hy + hz * hz);
            const long long num = (long long)N * s2 - ((long long)sx * sx + (long long)sy * sy + (long long)sz * sz);
            r.rg2 = (double)num / ((double)N * (double)N);
        }
        r.steps = alive ? (uint32_t)(N - 1) : dead;
        r.alive = alive ? 1u : 0u;
        r.digest = dg;
        p.rec[idx] = r;
    }
}

template <int Z, bool TRAJ, bool CONTACTS>
int launch_variant_c(const ModelParams& p, cudaStream_t stream)
{
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    const size_t fixed = (32 + 2 * Z) * sizeof(uint64_t);
    int threads = 256;
    while (threads > 32 && fixed + (size_t)p.N * 4 * threads > (size_t)(72 * 1024)) threads >>= 1;
    const size_t smem = fixed + (size_t)p.N * 4 * threads;
    auto kern = lattice_model_kernel<Z, TRAJ, CONTACTS>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -3;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) return -3;
    const uint64_t want = (p.n_chains + threads - 1) / threads, cap = (uint64_t)n_sm * per_sm;
    kern<<<(int)(want < cap ? want : cap), threads, smem, stream>>>(p);
    return cudaGetLastError() == cudaSuccess ? 1 : -3;
}

template <int Z, bool TRAJ>
int launch_variant(const ModelParams& p, cudaStream_t stream)
{
    bool flat = true;                   // all factors equal (q = 1): contact counts are irrelevant
    for (int c = 1; c < 32; ++c) flat = flat && p.Q[c] == p.Q[0];
    return flat ? launch_variant_c<Z, TRAJ, false>(p, stream) : launch_variant_c<Z, TRAJ, true>(p, stream);
}

}  // namespace

int launch_lattice_model(const ModelParams& p, cudaStream_t stream, const char** kernel_name)
{
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    int rc;
    if (p.z == 6) {
        *kernel_name = traj ? "lattice_model_kernel<z=6,traj>" : "lattice_model_kernel<z=6>";
        rc = traj ? launch_variant<6, true>(p, stream) : launch_variant<6, false>(p, stream);
    } else {
        *kernel_name = traj ? "lattice_model_kernel<z=26,traj>" : "lattice_model_kernel<z=26>";
        rc = traj ? launch_variant<26, true>(p, stream) : launch_variant<26, false>(p, stream);
    }
    if (rc < 0) return rc;
    const int rr = launch_reduce_records(p.rec, p.n_chains, p.chunk, p.n_vblocks, 0.0, p.lmax, p.out, p.partials, stream);
    return rr < 0 ? rr : rc + rr;
}

}  // namespace rosen
