// lattice.cu -- cubic-lattice Rosenbluth chain generation for sm_100a (steps L0-L5 of DESIGN.md 2;
// PAPER.md:88-179, Algorithm 1; weight Eq. 3 :58). One thread grows one chain at a time; the chain
// lives in shared memory as packed words split by monomer parity, because on a bipartite lattice
// only monomers j with j = s (mod 2) can sit next to the growth point r_{s-1}: the scan of
// Alg. 1 lines 13-17 / 26-31 touches floor(s/2) words instead of s-1 (exactly the same decisions).
#include <algorithm>
#include <math_constants.h>
#include "common.cuh"
#include "philox.cuh"
#include "reduce.cuh"

namespace rosen {

namespace {

// ---- packed site coordinates, 10-bit fields biased by 512 (|x| <= 511 => N <= 512) ------------------
constexpr uint32_t kBias   = 512u;
constexpr uint32_t kOrigin = kBias | (kBias << 10) | (kBias << 20);
constexpr uint32_t kDX = 1u, kDY = 1u << 10, kDZ = 1u << 20;

struct LatTables {
    uint32_t lut[64];   // index = occupied-direction mask; bits 0-2 = m, bits 3+3i.. = i-th free direction
    int4     step[8];   // per direction: {packed delta, dx, dy, dz}
    double   ln_m[8];   // ln m; ln_m[0] = -inf (dead)
};

__device__ __forceinline__ void build_tables(LatTables* t)
{
    for (int occ = threadIdx.x; occ < 64; occ += blockDim.x) {
        uint32_t e = 0, m = 0;
        for (int d = 0; d < 6; ++d)
            if (!((occ >> d) & 1)) { e |= (uint32_t)d << (3 + 3 * m); ++m; }
        t->lut[occ] = e | m;
    }
    if (threadIdx.x < 8) {
        const int d = threadIdx.x;
        const int ax = d >> 1, sg = (d & 1) ? -1 : 1;
        int4 s = make_int4(0, 0, 0, 0);
        if (d < 6) {
            s.x = sg * (int)(1u << (10 * ax));
            s.y = ax == 0 ? sg : 0; s.z = ax == 1 ? sg : 0; s.w = ax == 2 ? sg : 0;
        }
        t->step[d] = s;
        t->ln_m[d] = d == 0 ? -CUDART_INF : log((double)d);
    }
}

__device__ __forceinline__ uint64_t digest_fold(uint64_t h, uint32_t m, uint32_t choice)
{
    return (h ^ (uint64_t)(m | (choice << 8))) * 0x100000001B3ull;
}

// stride (in 32-bit words) of one thread's chain storage: two parity arrays of half4 words each,
// plus 4 words so that stride/4 is odd and LDS.128 of a quarter-warp is bank-conflict free.
__host__ __device__ inline int half4_of(int N) { return (((N + 1) / 2) + 3) & ~3; }
__host__ __device__ inline int stride_of(int N) { return 2 * half4_of(N) + 4; }

template <bool DIGEST, bool TRAJ>
__global__ void __launch_bounds__(256) lattice_int_kernel(const LatticeParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    LatTables* tab = reinterpret_cast<LatTables*>(smem_raw);
    Partial* scratch = reinterpret_cast<Partial*>(smem_raw + sizeof(LatTables));
    uint32_t* chains = reinterpret_cast<uint32_t*>(smem_raw + sizeof(LatTables) + 8 * sizeof(Partial));

    const int N = p.N;
    const int half4 = half4_of(N), stride = stride_of(N);
    uint32_t* ev = chains + (size_t)threadIdx.x * stride;   // monomers 0,2,4,...
    uint32_t* od = ev + half4;                              // monomers 1,3,5,...

    build_tables(tab);
    __syncthreads();

    Partial acc = partial_zero();
    const uint64_t nthreads = (uint64_t)gridDim.x * blockDim.x;

    for (uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < p.n_chains; idx += nthreads) {
        const uint64_t chain = p.chain_offset + idx;
        const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);

        // L0: r_0 = origin, lnW = 0, alive. Unused words hold 0, which no neighbour word can equal.
        for (int i = 0; i < stride / 4; ++i) reinterpret_cast<uint4*>(ev)[i] = make_uint4(0, 0, 0, 0);
        ev[0] = kOrigin;
        uint32_t h = kOrigin;
        int hx = 0, hy = 0, hz = 0, sx = 0, sy = 0, sz = 0, s2 = 0;
        double lnW = 0.0;
        bool alive = true;
        uint32_t steps = 0;
        uint64_t dg = 0xCBF29CE484222325ull;
        uint8_t* mrow = TRAJ && p.out.m_seq ? p.out.m_seq + idx * (uint64_t)(N - 1) : nullptr;

        for (int q = 0; 4 * q < N; ++q) {
            uint32_t w[4];
            philox4x32_10(c_lo, c_hi, (uint32_t)q, 0u, p.key0, p.key1, w);   // L1: one block per 4 steps
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int s = 4 * q + k;
                if (s == 0 || s >= N) continue;

                // L2: which of the 6 neighbours of r_{s-1} are occupied by r_j, j = s-2, s-4, ...
                const uint32_t n0 = h + kDX, n1 = h - kDX, n2 = h + kDY, n3 = h - kDY, n4 = h + kDZ, n5 = h - kDZ;
                bool o0 = false, o1 = false, o2 = false, o3 = false, o4 = false, o5 = false;
                const uint4* A = reinterpret_cast<const uint4*>((s & 1) ? od : ev);
                const int iters = ((s >> 1) + 3) >> 2;
                for (int i = 0; i < iters; ++i) {
                    const uint4 v = A[i];
                    o0 |= (v.x == n0); o1 |= (v.x == n1); o2 |= (v.x == n2); o3 |= (v.x == n3); o4 |= (v.x == n4); o5 |= (v.x == n5);
                    o0 |= (v.y == n0); o1 |= (v.y == n1); o2 |= (v.y == n2); o3 |= (v.y == n3); o4 |= (v.y == n4); o5 |= (v.y == n5);
                    o0 |= (v.z == n0); o1 |= (v.z == n1); o2 |= (v.z == n2); o3 |= (v.z == n3); o4 |= (v.z == n4); o5 |= (v.z == n5);
                    o0 |= (v.w == n0); o1 |= (v.w == n1); o2 |= (v.w == n2); o3 |= (v.w == n3); o4 |= (v.w == n4); o5 |= (v.w == n5);
                }
                const uint32_t occ = (uint32_t)o0 | ((uint32_t)o1 << 1) | ((uint32_t)o2 << 2) | ((uint32_t)o3 << 3) |
                                     ((uint32_t)o4 << 4) | ((uint32_t)o5 << 5);
                const uint32_t e = tab->lut[occ];
                const uint32_t m = e & 7u;

                // L3: weight. ln_m[0] = -inf makes a dead chain's lnW -inf for good.
                steps += alive ? 1u : 0u;
                lnW += tab->ln_m[m];
                if (TRAJ && mrow) mrow[s - 1] = alive ? (uint8_t)m : (uint8_t)0;

                // L4: uniform choice among the free neighbours, then place monomer s
                const uint32_t sel = __umulhi(w[k], m);
                const uint32_t dir = (e >> (3u + 3u * sel)) & 7u;
                if (DIGEST) { if (alive) dg = digest_fold(dg, m, m ? dir : 0xFFu); }
                alive = alive && (m != 0u);
                const int4 st = tab->step[dir];
                h += (uint32_t)st.x; hx += st.y; hy += st.z; hz += st.w;
                ((s & 1) ? od : ev)[s >> 1] = h;

                // L5: running sums for Rg^2
                sx += hx; sy += hy; sz += hz; s2 += hx * hx + hy * hy + hz * hz;
            }
        }

        // L5: per-chain observables (integers until the final divide)
        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            ree2 = (double)(hx * hx + hy * hy + hz * hz);
            const long long num = (long long)N * s2 - ((long long)sx * sx + (long long)sy * sy + (long long)sz * sz);
            rg2 = (double)num / ((double)N * (double)N);
        }
        const double wgt = alive ? exp(lnW - p.ln_shift) : 0.0;
        acc.sum_w += wgt; acc.sum_w_ree2 += wgt * ree2; acc.sum_w_rg2 += wgt * rg2; acc.sum_w2 += wgt * wgt;
        acc.n_dead += alive ? 0u : 1u; acc.n_steps += steps;
        if (DIGEST) { acc.digest_xor ^= dg; acc.digest_sum += dg; }

        if (p.out.lnW) p.out.lnW[idx] = lnW;
        if (p.out.alive) p.out.alive[idx] = alive ? 1 : 0;
        if (p.out.ree2) p.out.ree2[idx] = ree2;
        if (p.out.rg2) p.out.rg2[idx] = rg2;
        if (DIGEST && p.out.digest) p.out.digest[idx] = dg;
        if (TRAJ && p.out.conf) {
            // D1 (first version): each thread unpacks and writes its own chain; monomers from the
            // death step on are zero. steps = death step for a dead chain.
            int32_t* c = reinterpret_cast<int32_t*>(p.out.conf) + idx * (uint64_t)N * 3;
            const int placed = alive ? N : (int)steps;
            for (int i = 0; i < N; ++i) {
                const uint32_t v = ((i & 1) ? od : ev)[i >> 1];
                const bool ok = i < placed;
                c[3 * i + 0] = ok ? (int)(v & 1023u) - (int)kBias : 0;
                c[3 * i + 1] = ok ? (int)((v >> 10) & 1023u) - (int)kBias : 0;
                c[3 * i + 2] = ok ? (int)((v >> 20) & 1023u) - (int)kBias : 0;
            }
        }
    }

    block_reduce_store(acc, scratch, p.partials + blockIdx.x);
}

template <bool DIGEST, bool TRAJ>
int launch_int(const LatticeParams& p, cudaStream_t stream, int* grid_out)
{
    int dev = 0, n_sm = 0, smem_max = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    int smem_sm = 0;
    cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    const size_t fixed = sizeof(LatTables) + 8 * sizeof(Partial);
    const size_t per_thread = (size_t)stride_of(p.N) * 4;
    int threads = 256;
    while (threads > 32 && fixed + per_thread * threads > (size_t)(72 * 1024)) threads >>= 1;
    const size_t smem = fixed + per_thread * threads;
    if (smem > (size_t)smem_max) return -2;
    auto kern = lattice_int_kernel<DIGEST, TRAJ>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -3;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) return -3;
    // The grid (hence the reduction tree) must not depend on the output variant: size it from the
    // shared-memory / thread limits only, which are the same for every instantiation.
    per_sm = (int)std::min<size_t>(2048 / threads, (size_t)(smem_sm - 1024) / (smem + 1024));
    if (per_sm < 1) per_sm = 1;
    uint64_t want = (p.n_chains + threads - 1) / threads;
    uint64_t cap = (uint64_t)n_sm * per_sm;
    if (cap > (uint64_t)kMaxPartials) cap = kMaxPartials;
    const int grid = (int)(want < cap ? want : cap);
    kern<<<grid, threads, smem, stream>>>(p);
    if (cudaGetLastError() != cudaSuccess) return -3;
    *grid_out = grid;
    return 1;
}

}  // namespace

int launch_lattice(const LatticeParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    if (traj) {
        *kernel_name = digest ? "lattice_int_kernel<digest,traj>" : "lattice_int_kernel<traj>";
        return digest ? launch_int<true, true>(p, stream, grid_out) : launch_int<false, true>(p, stream, grid_out);
    }
    *kernel_name = digest ? "lattice_int_kernel<digest>" : "lattice_int_kernel<>";
    return digest ? launch_int<true, false>(p, stream, grid_out) : launch_int<false, false>(p, stream, grid_out);
}

}  // namespace rosen
