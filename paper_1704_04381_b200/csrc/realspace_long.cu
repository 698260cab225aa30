// realspace_long.cu -- off-lattice Rosenbluth generation for LONG chains (400 <= N <= 16383), the range of the paper's
// real-space "global-memory version" (Table 2: N = 100 ... 10000; Fig. 2b, :296). Same steps R0-R5,
// the same fp32 arithmetic and therefore the same decisions as realspace.cu, but the chain lives in HBM
// and the O(s) candidate scan of each step is replaced by a per-chain CELL LIST, so a chain costs O(N k) instead of
// O(N^2): only monomers in the 27 cells around the growth point can lie inside the candidate radius.
//
// Layout. One warp grows one chain. Per warp, in HBM:
//   float4   r[n_pad]            the chain: (x, y, z, link), link = bits of the index of the monomer placed before this one
//                                in the same cell (0xFFFF: none) -- one 16-byte load per hop of a list walk
//   entry    table[entries]      open-addressed map cell -> most recent monomer in it: 16 bytes,
//                                .x = (cx+2^14) | (cy+2^14) << 15 | (cz+2^14) << 30 | generation << 45, .y = monomer index
// cell = floor(coordinate * inv_cell) with cell edge = candidate radius x (1 + 2^-6): the slack covers the fp32
// rounding of the product (|x| <= 16383 b: error < 2^-9 cells), so |x_j - x_h| < radius implies cells differ by <= 1.
// Entries of another generation are empty (the counter is kept across calls: one memset per allocation or layout change); entries >= N + 1 > cells a chain can touch.
// Lanes 0..26 look up the 27 cells together and walk their lists in lock step; monomers that pass the candidate test
// of realspace.cu are compacted into a shared-memory buffer, which is flushed through the trial tests whenever it
// fills (overlap is an OR over candidates, so batching and order do not matter).
//
// Warps draw chains from a global ticket and write one record per chain; reduce_records_kernel (lattice_hash.cu)
// forms the deterministic sums afterwards, exactly as for the long lattice chains.
#include <cstdlib>
#include <math_constants.h>
#include "common.cuh"
#include "direction.cuh"
#include "philox.cuh"

namespace rosen {

namespace {

constexpr int      kCellField = 15;
constexpr int      kCellBias = 1 << (kCellField - 1);
constexpr int      kGenShift = 3 * kCellField;                       // 45
constexpr uint32_t kGenMax = (1u << (64 - kGenShift)) - 1u;
constexpr uint32_t kNone = 0xFFFFu;
constexpr int      kCandCap = (int)kRealLongCandCap;                 // float4 candidates buffered per warp
constexpr int      kWarpsPerBlock = 8;

__device__ __forceinline__ uint32_t slot_of(uint64_t key, uint32_t entries)
{
    return __umulhi((uint32_t)((key * 0x9E3779B97F4A7C15ull) >> 32), entries);
}

__device__ __forceinline__ uint64_t cell_key(int cx, int cy, int cz)
{
    return (uint64_t)(uint32_t)(cx + kCellBias) | ((uint64_t)(uint32_t)(cy + kCellBias) << kCellField) |
           ((uint64_t)(uint32_t)(cz + kCellBias) << (2 * kCellField));
}

// R2 for one batch of candidates: every trial of this lane against cand[0..n)
template <int PP, int E>
__device__ __forceinline__ void test_batch(const float4* cand, int n, const float (&tx)[PP][E], const float (&ty)[PP][E],
                                           const float (&tz)[PP][E], bool (&fr)[PP][E], float sigma2)
{
    for (int c = 0; c < n; ++c) {
        const float4 rj = cand[c];
#pragma unroll
        for (int pp = 0; pp < PP; ++pp)
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const float dx = __fsub_rn(rj.x, tx[pp][e]), dy = __fsub_rn(rj.y, ty[pp][e]), dz = __fsub_rn(rj.z, tz[pp][e]);
                const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                if (d2 < sigma2) fr[pp][e] = false;
            }
    }
}

// P = Philox blocks (trial pairs) per lane: lane owns trials 2 (lane + 32 pp) + {0, 1}. P = 0 (k <= 32): ONE trial per lane,
// trial t = lane from block lane >> 1 (the pair's two lanes draw the same block), so that 16 trials keep 16 lanes busy.
template <int P, bool DIGEST, bool TRAJ>
__global__ void __launch_bounds__(32 * kWarpsPerBlock) realspace_long_kernel(const RealLongParams p)
{
    constexpr int PP = P == 0 ? 1 : P, E = P == 0 ? 1 : 2;
    __shared__ double ln_tab[256];
    __shared__ float4 cand_all[kWarpsPerBlock][kCandCap];
    for (int i = threadIdx.x; i < 256; i += blockDim.x) ln_tab[i] = i == 0 ? -CUDART_INF : log((double)i);
    __syncthreads();

    const int N = p.N, k = p.k;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t below = (1u << lane) - 1u;
    const uint32_t entries = p.entries;
    float4* cand = cand_all[warp];
    unsigned char* base = p.work + ((uint64_t)blockIdx.x * kWarpsPerBlock + warp) * p.warp_bytes;
    float4* R4 = reinterpret_cast<float4*>(base);
    ulonglong2* table = reinterpret_cast<ulonglong2*>(base + (size_t)p.n_pad * 16);
    // this lane's cell offset among the 27 (lanes 27..31 idle in the look-up)
    const int ox = lane % 3 - 1, oy = (lane / 3) % 3 - 1, oz = lane / 9 - 1;
    const uint64_t gwarp = (uint64_t)blockIdx.x * kWarpsPerBlock + warp;
    uint32_t gen = p.gen_store[gwarp];      // generations continue across calls of one workspace layout (no memset per call)

    for (;;) {
        // ---- the warp draws its next chain (timing dependent; the record is a function of the chain id only)
        unsigned long long idx = 0;
        if (lane == 0) idx = atomicAdd(p.ticket, 1ull);
        idx = __shfl_sync(0xffffffffu, idx, 0);
        if (idx >= p.n_chains) { if (lane == 0) p.gen_store[gwarp] = gen; break; }
        const uint64_t chain = p.chain_offset + idx;
        const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);
        if (++gen > kGenMax) {
            for (uint32_t i = lane; i < entries; i += 32) table[i] = make_ulonglong2(0ull, 0ull);
            __syncwarp();                   // every lane's clears land before lane 0 enters the origin's cell below
            gen = 1u;
        }
        const uint64_t tag = (uint64_t)gen << kGenShift;

        // ---- R0: r_0 = origin, alone in its cell
        float hx = 0.f, hy = 0.f, hz = 0.f;
        if (lane == 0) {
            R4[0] = make_float4(0.f, 0.f, 0.f, __uint_as_float(kNone));
            const uint64_t key0 = cell_key(0, 0, 0);
            table[slot_of(key0, entries)] = make_ulonglong2(key0 | tag, 0ull);
        }
        double lnW = 0.0, Sx = 0.0, Sy = 0.0, Sz = 0.0, S2 = 0.0;
        uint32_t dead = 0;
        uint64_t dg = 0xCBF29CE484222325ull;
        uint32_t selw[4] = {0, 0, 0, 0};
        uint8_t* mrow = TRAJ && p.out.m_seq ? p.out.m_seq + idx * (uint64_t)(N - 1) : nullptr;
        __syncwarp();

        int s = 1;
        for (; s < N; ++s) {
            if ((s & 3) == 0 || s == 1) philox4x32_10(c_lo, c_hi, (uint32_t)(s >> 2), 0u, p.key0, p.key1, selw);
            const uint32_t usel = (s & 2) ? ((s & 1) ? selw[3] : selw[2]) : ((s & 1) ? selw[1] : selw[0]);

            // ---- R1: this lane's trials (P Philox blocks = 2P trials), trial index t = 2 (lane + 32 pp) + e
            float tx[PP][E], ty[PP][E], tz[PP][E];
            bool fr[PP][E];
#pragma unroll
            for (int pp = 0; pp < PP; ++pp) {
                const uint32_t bi = P == 0 ? (uint32_t)lane >> 1 : (uint32_t)(lane + 32 * pp);
                uint32_t w[4];
                philox4x32_10(c_lo, c_hi, (uint32_t)s, 1u + bi, p.key0, p.key1, w);
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const bool second = P == 0 ? (lane & 1) != 0 : e != 0;       // which trial of the pair
                    float ux, uy, uz;
                    direction(second ? w[2] : w[0], second ? w[3] : w[1], ux, uy, uz);
                    tx[pp][e] = __fmaf_rn(p.b, ux, hx);
                    ty[pp][e] = __fmaf_rn(p.b, uy, hy);
                    tz[pp][e] = __fmaf_rn(p.b, uz, hz);
                    fr[pp][e] = (int)(2u * bi + (second ? 1u : 0u)) < k;
                }
            }

            // ---- R2: candidates = monomers j <= s-2 inside the candidate radius of r_{s-1}, from the 27 cells around it
            const int hcx = __float2int_rd(__fmul_rn(hx, p.inv_cell)), hcy = __float2int_rd(__fmul_rn(hy, p.inv_cell)),
                      hcz = __float2int_rd(__fmul_rn(hz, p.inv_cell));
            uint32_t node = kNone;
            if (lane < 27) {
                const uint64_t want = cell_key(hcx + ox, hcy + oy, hcz + oz) | tag;
                uint32_t sl = slot_of(want & ~(~0ull << kGenShift), entries);
                for (;;) {
                    const ulonglong2 e = table[sl];
                    if ((uint32_t)(e.x >> kGenShift) != gen) break;                 // empty: no monomer in this cell
                    if (e.x == want) { node = (uint32_t)e.y; break; }
                    sl = sl + 1u == entries ? 0u : sl + 1u;
                }
            }
            int ncand = 0;
            while (__any_sync(0xffffffffu, node != kNone)) {
                bool in = false;
                float4 rj = make_float4(0.f, 0.f, 0.f, 0.f);
                if (node != kNone) {
                    rj = R4[node];
                    const uint32_t nx = __float_as_uint(rj.w);
                    const float ax = rj.x - hx, ay = rj.y - hy, az = rj.z - hz;
                    in = (int)node < s - 1 && fmaf(az, az, fmaf(ay, ay, ax * ax)) < p.prefilter2;
                    node = nx;
                }
                const uint32_t bal = __ballot_sync(0xffffffffu, in);
                if (in) cand[ncand + __popc(bal & below)] = rj;
                ncand += __popc(bal);
                if (ncand > (int)p.cand_cap - 32) {    // buffer may not hold another round: test what is there
                    __syncwarp();
                    test_batch<PP, E>(cand, ncand, tx, ty, tz, fr, p.sigma2);
                    ncand = 0;
                    __syncwarp();
                }
            }
            __syncwarp();
            test_batch<PP, E>(cand, ncand, tx, ty, tz, fr, p.sigma2);

            // ---- m_s and the rank of each free trial in trial order
            uint32_t B[PP][E];
            uint32_t m = 0;
#pragma unroll
            for (int pp = 0; pp < PP; ++pp)
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    B[pp][e] = __ballot_sync(0xffffffffu, fr[pp][e]);
                    m += __popc(B[pp][e]);
                }
            if (TRAJ && mrow && lane == 0) mrow[s - 1] = (uint8_t)m;

            // ---- R3
            if (m == 0u) { dead = (uint32_t)s; if (DIGEST) dg = digest_fold(dg, 0u, 0xFFu); break; }
            lnW += ln_tab[m];

            // ---- R4: the sel-th free trial (in trial order) becomes r_s
            const uint32_t sel = __umulhi(usel, m);
            uint32_t rank0 = 0;
            bool hit = false;
            float px = hx, py = hy, pz = hz;
            uint32_t tsel = 0;
#pragma unroll
            for (int pp = 0; pp < PP; ++pp) {
                if (P == 0) {
                    if (fr[0][0] && (uint32_t)__popc(B[0][0] & below) == sel) { hit = true; px = tx[0][0]; py = ty[0][0]; pz = tz[0][0]; tsel = (uint32_t)lane; }
                } else {
                    const uint32_t r0 = rank0 + __popc(B[pp][0] & below) + __popc(B[pp][E - 1] & below);
                    const uint32_t r1 = r0 + (fr[pp][0] ? 1u : 0u);
                    if (fr[pp][0] && r0 == sel) { hit = true; px = tx[pp][0]; py = ty[pp][0]; pz = tz[pp][0]; tsel = 2u * (lane + 32 * pp); }
                    if (fr[pp][E - 1] && r1 == sel) { hit = true; px = tx[pp][E - 1]; py = ty[pp][E - 1]; pz = tz[pp][E - 1]; tsel = 2u * (lane + 32 * pp) + 1u; }
                    rank0 += __popc(B[pp][0]) + __popc(B[pp][E - 1]);
                }
            }
            const uint32_t hb = __ballot_sync(0xffffffffu, hit);
            const int src = __ffs(hb) - 1;
            hx = __shfl_sync(0xffffffffu, px, src); hy = __shfl_sync(0xffffffffu, py, src);
            hz = __shfl_sync(0xffffffffu, pz, src); tsel = __shfl_sync(0xffffffffu, tsel, src);
            if (DIGEST) dg = digest_fold(dg, m, tsel);

            // store r_s and push it on its cell's list (lane 0; the warp sees it after the __syncwarp)
            if (lane == 0) {
                const uint64_t want = cell_key(__float2int_rd(__fmul_rn(hx, p.inv_cell)), __float2int_rd(__fmul_rn(hy, p.inv_cell)),
                                               __float2int_rd(__fmul_rn(hz, p.inv_cell))) | tag;
                uint32_t sl = slot_of(want & ~(~0ull << kGenShift), entries);
                uint32_t prev = kNone;
                for (;;) {
                    const ulonglong2 e = table[sl];
                    if ((uint32_t)(e.x >> kGenShift) != gen) break;                 // empty: first monomer of this cell
                    if (e.x == want) { prev = (uint32_t)e.y; break; }
                    sl = sl + 1u == entries ? 0u : sl + 1u;
                }
                R4[s] = make_float4(hx, hy, hz, __uint_as_float(prev));
                table[sl] = make_ulonglong2(want, (uint64_t)s);
            }

            // ---- R5 running sums (fp64)
            Sx += (double)hx; Sy += (double)hy; Sz += (double)hz;
            S2 += (double)hx * (double)hx + (double)hy * (double)hy + (double)hz * (double)hz;
            __syncwarp();
        }

        const bool alive = dead == 0u;
        const uint32_t steps = alive ? (uint32_t)(N - 1) : dead;
        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            ree2 = (double)hx * (double)hx + (double)hy * (double)hy + (double)hz * (double)hz;
            const double inv = 1.0 / (double)N;
            const double cx = Sx * inv, cy = Sy * inv, cz = Sz * inv;
            rg2 = S2 * inv - (cx * cx + cy * cy + cz * cz);
        }
        if (lane == 0) {
            ChainRecord r;
            r.lnW = alive ? lnW : -CUDART_INF; r.ree2 = ree2; r.rg2 = rg2;
            r.steps = steps; r.alive = alive ? 1u : 0u; r.digest = DIGEST ? dg : 0ull;
            p.rec[idx] = r;
        }
        if (TRAJ) {
            // D1: the warp streams its chain from its HBM region to [N][3], zeros from the death step on (reading A13)
            __syncwarp();
            const int placed = alive ? N : (int)steps;
            if (p.out.conf) {
                float* c = reinterpret_cast<float*>(p.out.conf) + idx * (uint64_t)N * 3;
                for (int e = lane; e < 3 * N; e += 32) {
                    const int i = e / 3, a = e - 3 * i;
                    c[e] = i < placed ? reinterpret_cast<const float*>(R4)[4 * i + a] : 0.0f;
                }
            }
            if (mrow) for (int e = (int)steps + lane; e < N - 1; e += 32) mrow[e] = 0;
        }
        __syncwarp();
    }
}

template <int P, bool DIGEST, bool TRAJ>
int launch_variant(const RealLongParams& p, int n_warps, cudaStream_t stream)
{
    realspace_long_kernel<P, DIGEST, TRAJ><<<n_warps / kWarpsPerBlock, 32 * kWarpsPerBlock, 0, stream>>>(p);
    return cudaGetLastError() == cudaSuccess ? 1 : -3;
}

template <int P>
int launch_p(const RealLongParams& p, int n_warps, cudaStream_t stream)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    if (traj) return digest ? launch_variant<P, true, true>(p, n_warps, stream) : launch_variant<P, false, true>(p, n_warps, stream);
    return digest ? launch_variant<P, true, false>(p, n_warps, stream) : launch_variant<P, false, false>(p, n_warps, stream);
}

}  // namespace

uint32_t real_long_gen_max() { return kGenMax; }

int real_long_max_warps(int k, int* warps_out)
{
    int dev = 0, n_sm = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    cudaError_t e;
    if (k <= 32)       e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, realspace_long_kernel<0, true, true>, 32 * kWarpsPerBlock, 0);
    else if (k <= 64)  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, realspace_long_kernel<1, true, true>, 32 * kWarpsPerBlock, 0);
    else if (k <= 128) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, realspace_long_kernel<2, true, true>, 32 * kWarpsPerBlock, 0);
    else               e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, realspace_long_kernel<4, true, true>, 32 * kWarpsPerBlock, 0);
    if (e != cudaSuccess || per_sm < 1) return -3;
    *warps_out = n_sm * per_sm * kWarpsPerBlock;
    return 0;
}

int launch_realspace_long(const RealLongParams& p, int n_warps, cudaStream_t stream, const char** kernel_name)
{
    int rc;
    if (p.k <= 32)       { *kernel_name = "realspace_long_kernel<P=1/2>"; rc = launch_p<0>(p, n_warps, stream); }
    else if (p.k <= 64)  { *kernel_name = "realspace_long_kernel<P=1>"; rc = launch_p<1>(p, n_warps, stream); }
    else if (p.k <= 128) { *kernel_name = "realspace_long_kernel<P=2>"; rc = launch_p<2>(p, n_warps, stream); }
    else                 { *kernel_name = "realspace_long_kernel<P=4>"; rc = launch_p<4>(p, n_warps, stream); }
    if (rc < 0) return rc;
    rc = launch_reduce_records(p.rec, p.n_chains, p.chunk, p.n_vblocks, p.ln_shift, p.lmax, p.out, p.partials, stream);
    return rc < 0 ? rc : 1 + rc;
}

}  // namespace rosen
