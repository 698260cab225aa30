// realspace.cu -- off-lattice Rosenbluth chain generation for sm_100a (steps R0-R5 of DESIGN.md 2;
// PAPER.md:185-187 sec. 3.3.3, :202-262 Algorithm 2). A group of G lanes grows one chain: lane =
// pair of trials (one Philox block), so the trial loop of Alg. 2 line 9 runs across lanes and the
// free-trial count is a __ballot_sync/__popc. The chain lives in shared memory (SoA fp32).
//
// Exact pruning of Alg. 2 lines 13-19: a monomer farther than (b + sigma)(1 + 2^-9) from the growth
// point r_{s-1} cannot be within sigma of any trial (every trial is b(1 +- 1e-6) away from r_{s-1}),
// so each step first collects the few candidates inside that radius (cooperatively, lanes =
// monomers) and tests the trials against those only. Decisions are identical to the full scan;
// the argument with its fp32 error budget is DESIGN.md 5.2.
//
// All fp32 arithmetic that decides anything is written with explicit __f*_rn intrinsics in the order
// DESIGN.md 3.3 fixes, so nvcc cannot contract or reorder it.
#include <algorithm>
#include <math_constants.h>
#include "common.cuh"
#include "direction.cuh"
#include "philox.cuh"
#include "reduce.cuh"

namespace rosen {

namespace {

// shared memory carve-up (bytes) -----------------------------------------------------------------
//   double   ln_tab[256]            ln m, ln_tab[0] = -inf
//   Partial  scratch[32]
//   per group: float4 r[Np] (x, y, z, unused); uint16 cand[Np] (byte offsets into r); uint8 mseq[Np]   (Np = N rounded up to 4)
__host__ __device__ inline int n_pad(int N) { return (N + 3) & ~3; }
__host__ __device__ inline size_t group_bytes(int N) { return (size_t)n_pad(N) * (16 + 2 + 1) + 4; }

template <int G, int P, bool DIGEST, bool TRAJ>
__global__ void __launch_bounds__(256, TRAJ ? 3 : 0) realspace_kernel(const RealParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* ln_tab = reinterpret_cast<double*>(smem_raw);
    Partial* scratch = reinterpret_cast<Partial*>(smem_raw + 256 * sizeof(double));
    unsigned char* gbase_ptr = smem_raw + 256 * sizeof(double) + 32 * sizeof(Partial);

    const int N = p.N, k = p.k, Np = n_pad(N);
    const int lane = threadIdx.x & 31;
    const int gl = lane & (G - 1);                         // lane within the group
    const int gshift = lane & ~(G - 1);                    // first lane of the group in the warp
    const uint32_t gmask = (G == 32) ? 0xffffffffu : ((1u << G) - 1u);
    const uint32_t below = (1u << gl) - 1u;
    const int group_in_block = threadIdx.x / G;
    const size_t gsz = (group_bytes(N) + 15) & ~(size_t)15;
    float4* R4 = reinterpret_cast<float4*>(gbase_ptr + gsz * group_in_block);   // one LDS.128 per monomer
    uint16_t* cand = reinterpret_cast<uint16_t*>(R4 + Np);
    uint8_t* mbuf = reinterpret_cast<uint8_t*>(cand + Np);

    for (int i = threadIdx.x; i < 256; i += blockDim.x) ln_tab[i] = i == 0 ? -CUDART_INF : log((double)i);
    __syncthreads();

    // Virtual blocks (common.cuh): virtual block vb owns chains [vb*chunk, (vb+1)*chunk); group g of the block takes
    // chains vb*chunk + it*gpb + g. Blocks draw virtual blocks from a ticket counter, so the grid only balances load.
    const uint32_t gpb = blockDim.x / G;                     // groups per block; chunk is a multiple of 256 >= gpb
    const uint32_t iters = p.chunk / gpb;                    // the same for every group of a warp (warp primitives below)
    __shared__ uint32_t vb_ticket;
    for (;;) {
    if (threadIdx.x == 0) vb_ticket = atomicAdd(p.vb_counter, 1u);
    __syncthreads();
    const uint32_t vb = vb_ticket;
    if (vb >= p.n_vblocks) break;
    Partial acc = partial_zero();

    for (uint32_t it = 0; it < iters; ++it) {
        const uint64_t idx = (uint64_t)vb * p.chunk + (uint64_t)it * gpb + (uint32_t)group_in_block;
        const bool active = idx < p.n_chains;               // inactive groups compute and discard
        const uint64_t chain = p.chain_offset + idx;
        const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);

        // R0
        float hx = 0.f, hy = 0.f, hz = 0.f;
        if (gl == 0) R4[0] = make_float4(0.f, 0.f, 0.f, 0.f);
        double lnW = 0.0, Sx = 0.0, Sy = 0.0, Sz = 0.0, S2 = 0.0;
        bool alive = true;
        uint32_t steps = 0;
        uint64_t dg = 0xCBF29CE484222325ull;
        uint32_t selw[4] = {0, 0, 0, 0};
        uint32_t usel = 0;
        __syncwarp();

        for (int s = 1; s < N; ++s) {
            if ((s & 3) == 0 || s == 1) philox4x32_10(c_lo, c_hi, (uint32_t)(s >> 2), 0u, p.key0, p.key1, selw);
            {   // word s & 3 without a dynamically indexed (local-memory) array
                const uint32_t lo = (s & 1) ? selw[1] : selw[0], hi = (s & 1) ? selw[3] : selw[2];
                usel = (s & 2) ? hi : lo;
            }

            // ---- candidates: monomers j <= s-2 within the conservative radius of r_{s-1}
            // (two monomers per lane and iteration: independent loads and distance chains hide each other's latency;
            // the order of the list is irrelevant, overlap is an OR over candidates)
            int ncand = 0;
            for (int j0 = 0; j0 < s - 1; j0 += 2 * G) {
                const int ja = j0 + gl, jb = ja + G;
                const float4 ra = R4[min(ja, s - 2)], rb = R4[min(jb, s - 2)];
                const float ax = ra.x - hx, ay = ra.y - hy, az = ra.z - hz;
                const float bx = rb.x - hx, by = rb.y - hy, bz = rb.z - hz;
                const bool ina = ja < s - 1 && fmaf(az, az, fmaf(ay, ay, ax * ax)) < p.prefilter2;
                const bool inb = jb < s - 1 && fmaf(bz, bz, fmaf(by, by, bx * bx)) < p.prefilter2;
                const uint32_t bita = (__ballot_sync(0xffffffffu, ina) >> gshift) & gmask;
                const uint32_t bitb = (__ballot_sync(0xffffffffu, inb) >> gshift) & gmask;
                const int na = __popc(bita);
                if (ina) cand[ncand + __popc(bita & below)] = (uint16_t)(ja * 16);
                if (inb) cand[ncand + na + __popc(bitb & below)] = (uint16_t)(jb * 16);
                ncand += na + __popc(bitb);
            }
            __syncwarp();

            // ---- R1 + R2: this lane's trials (P Philox blocks = 2P trials)
            float tx[P][2], ty[P][2], tz[P][2];
            bool fr[P][2];
#pragma unroll
            for (int pp = 0; pp < P; ++pp) {
                const uint32_t bi = (uint32_t)(gl + G * pp);
                uint32_t w[4];
                philox4x32_10(c_lo, c_hi, (uint32_t)s, 1u + bi, p.key0, p.key1, w);
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    float ux, uy, uz;
                    direction(w[2 * e], w[2 * e + 1], ux, uy, uz);
                    tx[pp][e] = __fmaf_rn(p.b, ux, hx);
                    ty[pp][e] = __fmaf_rn(p.b, uy, hy);
                    tz[pp][e] = __fmaf_rn(p.b, uz, hz);
                    fr[pp][e] = (int)(2u * bi + e) < k;
                }
            }
            for (int c = 0; c < ncand; ++c) {
                const float4 rj = *reinterpret_cast<const float4*>(reinterpret_cast<const unsigned char*>(R4) + cand[c]);
                const float xj = rj.x, yj = rj.y, zj = rj.z;
#pragma unroll
                for (int pp = 0; pp < P; ++pp)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const float dx = __fsub_rn(xj, tx[pp][e]), dy = __fsub_rn(yj, ty[pp][e]), dz = __fsub_rn(zj, tz[pp][e]);
                        const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                        if (d2 < p.sigma2) fr[pp][e] = false;
                    }
            }

            // ---- m_s and the rank of each free trial in trial order t = 2*(gl + G*pp) + e
            uint32_t B[P][2];
            uint32_t m = 0;
#pragma unroll
            for (int pp = 0; pp < P; ++pp)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    B[pp][e] = (__ballot_sync(0xffffffffu, fr[pp][e]) >> gshift) & gmask;
                    m += __popc(B[pp][e]);
                }

            // ---- R3
            steps += alive ? 1u : 0u;
            lnW += ln_tab[m];
            if (TRAJ) { if (gl == 0 && p.out.m_seq) mbuf[s - 1] = alive ? (uint8_t)m : (uint8_t)0; }

            // ---- R4: the sel-th free trial
            const uint32_t sel = __umulhi(usel, m);
            uint32_t base = 0;
            bool hit = false;
            float px = hx, py = hy, pz = hz;
            uint32_t tsel = 0;
#pragma unroll
            for (int pp = 0; pp < P; ++pp) {
                const uint32_t r0 = base + __popc(B[pp][0] & below) + __popc(B[pp][1] & below);
                const uint32_t r1 = r0 + (fr[pp][0] ? 1u : 0u);
                if (fr[pp][0] && r0 == sel) { hit = true; px = tx[pp][0]; py = ty[pp][0]; pz = tz[pp][0]; tsel = 2u * (gl + G * pp); }
                if (fr[pp][1] && r1 == sel) { hit = true; px = tx[pp][1]; py = ty[pp][1]; pz = tz[pp][1]; tsel = 2u * (gl + G * pp) + 1u; }
                base += __popc(B[pp][0]) + __popc(B[pp][1]);
            }
            const uint32_t hb = (__ballot_sync(0xffffffffu, hit) >> gshift) & gmask;
            const int src = gshift + (hb ? __ffs(hb) - 1 : 0);
            px = __shfl_sync(0xffffffffu, px, src); py = __shfl_sync(0xffffffffu, py, src);
            pz = __shfl_sync(0xffffffffu, pz, src); tsel = __shfl_sync(0xffffffffu, tsel, src);
            if (DIGEST) { if (alive) dg = digest_fold(dg, m, m ? tsel : 0xFFu); }
            alive = alive && (m != 0u);
            if (m != 0u) { hx = px; hy = py; hz = pz; }
            if (gl == 0) R4[s] = make_float4(hx, hy, hz, 0.f);

            // ---- R5 running sums (fp64)
            Sx += (double)hx; Sy += (double)hy; Sz += (double)hz;
            S2 += (double)hx * (double)hx + (double)hy * (double)hy + (double)hz * (double)hz;
            __syncwarp();
        }

        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            ree2 = (double)hx * (double)hx + (double)hy * (double)hy + (double)hz * (double)hz;
            const double inv = 1.0 / (double)N;
            const double cx = Sx * inv, cy = Sy * inv, cz = Sz * inv;
            rg2 = S2 * inv - (cx * cx + cy * cy + cz * cz);
        }
        const double wgt = alive ? exp(lnW - p.ln_shift) : 0.0;
        if (active && gl == 0) {
            acc.sum_w += wgt; acc.sum_w_ree2 += wgt * ree2; acc.sum_w_rg2 += wgt * rg2; acc.sum_w2 += wgt * wgt;
            acc.n_dead += alive ? 0u : 1u; acc.n_steps += steps;
            if (DIGEST) { acc.digest_xor ^= dg; acc.digest_sum += dg; }
            if (p.out.lnW) p.out.lnW[idx] = lnW;
            if (p.out.alive) p.out.alive[idx] = alive ? 1 : 0;
            if (p.out.ree2) p.out.ree2[idx] = ree2;
            if (p.out.rg2) p.out.rg2[idx] = rg2;
            if (DIGEST && p.out.digest) p.out.digest[idx] = dg;
        }
        if (TRAJ && active) {
            // D1: the group streams its chain out of shared memory, interleaving SoA -> [N][3]
            const int placed = alive ? N : (int)steps;
            if (p.out.conf) {
                float* c = reinterpret_cast<float*>(p.out.conf) + idx * (uint64_t)N * 3;
                for (int e = gl; e < 3 * N; e += G) {
                    const int i = e / 3, a = e - 3 * i;
                    const float v = reinterpret_cast<const float*>(R4)[4 * i + a];
                    c[e] = i < placed ? v : 0.0f;
                }
            }
            if (p.out.m_seq) {
                uint8_t* mr = p.out.m_seq + idx * (uint64_t)(N - 1);
                for (int e = gl; e < N - 1; e += G) mr[e] = mbuf[e];
            }
        }
        __syncwarp();
    }

    block_reduce_store(acc, scratch, p.partials + vb);
    }
}

template <int G, int P, bool DIGEST, bool TRAJ>
int launch_one(const RealParams& p, cudaStream_t stream, int* grid_out)
{
    int dev = 0, n_sm = 0, smem_max = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t fixed = 256 * sizeof(double) + 32 * sizeof(Partial);
    const size_t gsz = (group_bytes(p.N) + 15) & ~(size_t)15;
    int threads = 256;
    while (threads > 32 && fixed + gsz * (threads / G) > (size_t)(100 * 1024)) threads >>= 1;
    const size_t smem = fixed + gsz * (threads / G);
    if (smem > (size_t)smem_max) return -2;
    auto kern = realspace_kernel<G, P, DIGEST, TRAJ>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -3;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) return -3;
    // one resident wave of this variant; the sums do not depend on the grid (virtual blocks)
    uint64_t cap = (uint64_t)n_sm * per_sm;
    const int grid = (int)(p.n_vblocks < cap ? p.n_vblocks : cap);
    kern<<<grid, threads, smem, stream>>>(p);
    if (cudaGetLastError() != cudaSuccess) return -3;
    *grid_out = grid;
    return 1;
}

template <int G, int P>
int launch_gp(const RealParams& p, cudaStream_t stream, int* grid_out)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    if (traj) return digest ? launch_one<G, P, true, true>(p, stream, grid_out) : launch_one<G, P, false, true>(p, stream, grid_out);
    return digest ? launch_one<G, P, true, false>(p, stream, grid_out) : launch_one<G, P, false, false>(p, stream, grid_out);
}

}  // namespace

int launch_realspace(const RealParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out)
{
    int blocks = (p.k + 1) / 2;   // Philox blocks (trial pairs) per step
    // Long chains: a warp holds 32/G chains of group_bytes(N) each; widen the group (idle lanes own trials >= k)
    // until one warp's chains fit 24 KB, so that a block of >= 4 warps fits shared memory (N = 2048: one chain per warp, 2 warps per block).
    {
        const size_t gsz = (group_bytes(p.N) + 15) & ~(size_t)15;
        int g_mem = 1;
        while (g_mem < 32 && (32 / g_mem) * gsz > (size_t)(24 * 1024)) g_mem *= 2;
        if (g_mem > 4 && blocks < g_mem) blocks = g_mem;      // selects <G = g_mem, P = 1> below (g_mem = 8 -> G = 16)
        else if (g_mem > 1 && blocks < g_mem) blocks = g_mem; // 2 or 4
        if (g_mem == 8 && blocks <= 8) blocks = 9;            // no <8,1> variant: take <16,1>
    }
    if (blocks <= 1)  { *kernel_name = "realspace_kernel<G=1,P=1>";  return launch_gp<1, 1>(p, stream, grid_out); }
    if (blocks <= 2)  { *kernel_name = "realspace_kernel<G=2,P=1>";  return launch_gp<2, 1>(p, stream, grid_out); }
    if (blocks <= 4)  { *kernel_name = "realspace_kernel<G=4,P=1>";  return launch_gp<4, 1>(p, stream, grid_out); }
    // 5..8 blocks: 4 lanes x 2 blocks per lane measured 8 % faster than 8 x 1 (config 3: 41.5 -> 38.1 ms)
    if (blocks <= 8)  { *kernel_name = "realspace_kernel<G=4,P=2>";  return launch_gp<4, 2>(p, stream, grid_out); }
    if (blocks <= 16) { *kernel_name = "realspace_kernel<G=16,P=1>"; return launch_gp<16, 1>(p, stream, grid_out); }
    if (blocks <= 32) { *kernel_name = "realspace_kernel<G=32,P=1>"; return launch_gp<32, 1>(p, stream, grid_out); }
    if (blocks <= 64) { *kernel_name = "realspace_kernel<G=32,P=2>"; return launch_gp<32, 2>(p, stream, grid_out); }
    *kernel_name = "realspace_kernel<G=32,P=4>";
    return launch_gp<32, 4>(p, stream, grid_out);
}

}  // namespace rosen
