// realspace.cu -- off-lattice Rosenbluth chain generation for sm_100a (steps R0-R5 + D1 of DESIGN.md 2;
// PAPER.md:185-187 sec. 3.3.3, :202-262 Algorithm 2). A group of G lanes grows one chain: a lane owns 2P
// consecutive trials (P Philox blocks), so the trial loop of Alg. 2 line 9 runs across lanes. The chain lives
// in shared memory as float4 (x, y, z, -) per monomer, padded with far-away sentinels.
//
// Exact pruning of Alg. 2 lines 13-19: a monomer farther than (b + sigma)(1 + 2^-9) from the growth point
// r_{s-1} cannot be within sigma of any trial (every trial is b(1 +- 1e-6) away from r_{s-1}), so each step
// first marks the few candidates inside that radius -- 32 monomers per group and pass, one bit each -- and tests
// the trials against the marked monomers only. Decisions are identical to the full scan; the argument with its
// fp32 error budget is DESIGN.md 5.2.
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

constexpr size_t kFixedBytes = 256 * sizeof(double) + 32 * sizeof(Partial) + 32 * sizeof(uint64_t);   // ln_tab | scratch | Q
constexpr float kFar = 1.0e18f;   // sentinel coordinate: squared distances ~3e36 stay finite and fail every test

// shared memory carve-up (bytes) -----------------------------------------------------------------
//   double   ln_tab[256]            ln m, ln_tab[0] = -inf
//   Partial  scratch[32]
//   per group: float4 r[Np] (Np = N rounded up to 32; slots the chain has not reached hold the sentinel);
//              MSEQ variants: uint8 mseq[Np]
// The group stride is 16 G (mod 128) bytes for G <= 8, so that the groups of a quarter-warp reading G consecutive
// monomers each (LDS.128) cover all 32 banks once.
__host__ __device__ inline int n_pad(int N) { return (N + 31) & ~31; }
__host__ __device__ inline size_t group_bytes(int N, int G, bool mseq)
{
    size_t b = (size_t)n_pad(N) * (mseq ? 17 : 16);
    const size_t want = (size_t)(16 * G) % 128;
    b += (want + 128 - b % 128) % 128;
    return b;
}

__device__ __forceinline__ uint32_t bfind(uint32_t x)     // index of the most significant set bit (FLO.U32)
{
    uint32_t r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}

// t = |r - h|^2 - prefilter2 in one FFMA chain: negative (sign bit set) iff the monomer is inside the conservative radius
// (an exact zero rounds to +0). Its few-ulp rounding is covered by the radius margin like that of the plain sum.
__device__ __forceinline__ uint32_t inside_bits(const float4 r, float hx, float hy, float hz, float prefilter2)
{
    const float ax = r.x - hx, ay = r.y - hy, az = r.z - hz;
    return __float_as_uint(fmaf(az, az, fmaf(ay, ay, fmaf(ax, ax, -prefilter2))));
}

// ---- candidate bits of monomers [j0, j0 + 32) of this lane's group: bit i <=> |r_{j0+i} - h|^2 < prefilter2.
// base = R4 + j0; cnt = monomers left from j0 (>= 1, uniform over the warp). Slots beyond the scannable monomers hold the
// sentinel. Lane gl looks at slots G q + gl, q = 0 .. min(Q, ceil(cnt / G)) - 1.
template <int G>
__device__ __forceinline__ uint32_t candidate_bits(const float4* base, int cnt, int gl, int gshift, uint32_t gmask,
                                                   float hx, float hy, float hz, float pf)
{
    constexpr int Q = 32 / G;                 // monomers per lane and pass
    if constexpr (G == 32) {
        return __ballot_sync(0xffffffffu, (int32_t)inside_bits(base[gl], hx, hy, hz, pf) < 0);
    } else if constexpr (G >= 8) {
        uint32_t mask = 0;
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            if (G * q >= cnt) break;
            const uint32_t b = __ballot_sync(0xffffffffu, (int32_t)inside_bits(base[G * q + gl], hx, hy, hz, pf) < 0);
            mask |= ((b >> gshift) & gmask) << (G * q);
        }
        return mask;
    } else {
        uint32_t pm = 0;
        const float4* lb = base + gl;
#define ROSEN_PF(q) pm |= (inside_bits(lb[G * (q)], hx, hy, hz, pf) >> (31 - G * (q))) & (1u << (G * (q)));
        if constexpr (G == 4) {               // one computed jump per pass instead of a test per monomer
            switch ((cnt + 3) >> 2) {
                default: ROSEN_PF(7)
                case 7: ROSEN_PF(6)
                case 6: ROSEN_PF(5)
                case 5: ROSEN_PF(4)
                case 4: ROSEN_PF(3)
                case 3: ROSEN_PF(2)
                case 2: ROSEN_PF(1)
                case 1: ROSEN_PF(0)
            }
        } else {
#pragma unroll
            for (int q = 0; q < Q; ++q) {
                if (G * q >= cnt) break;
                ROSEN_PF(q)
            }
        }
#undef ROSEN_PF
        pm <<= gl;
#pragma unroll
        for (int d = 1; d < G; d <<= 1) pm |= __shfl_xor_sync(0xffffffffu, pm, d);
        return pm;
    }
}

// D1 store phase ("flushed to the global memory"): the group's lanes stream the chain out of shared memory,
// float4 (x, y, z, -) -> crow[N][3], zeros from monomer `placed` on. Rows are 12 N bytes: 16-byte aligned when N is a
// multiple of 4, then consecutive lanes store consecutive 16-byte pieces (G = 32: 512 contiguous bytes per instruction);
// otherwise 4-byte stores, still consecutive across lanes.
template <int G>
__device__ __forceinline__ void store_conf(const float4* R4, float* crow, int N, int placed, int gl)
{
    const float* Rf = reinterpret_cast<const float*>(R4);
    if ((N & 3) == 0) {
        float4* c4 = reinterpret_cast<float4*>(crow);
        for (int v = gl; v < 3 * (N >> 2); v += G) {
            float o[4];
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                const uint32_t e = 4u * (uint32_t)v + cc, i = (e * 43691u) >> 17;       // e / 3 for e < 98304
                o[cc] = (int)i < placed ? Rf[e + i] : 0.0f;                                // word 4 i + (e - 3 i)
            }
            c4[v] = make_float4(o[0], o[1], o[2], o[3]);
        }
    } else {
        for (int e = gl; e < 3 * N; e += G) {
            const uint32_t i = ((uint32_t)e * 43691u) >> 17;
            crow[e] = (int)i < placed ? Rf[e + i] : 0.0f;
        }
    }
}

// The store phase alone (rosen_realspace_dump_probe; SURVEY.md 8(d) "isolated store phase ... a dump-only kernel"): every
// group keeps one synthetic chain resident in shared memory and stores it, with store_conf above and the launch geometry
// of realspace_kernel<G, ...>, once per chain id of the call (+ one fp64 per chain, like lnW).
template <int G>
__global__ void __launch_bounds__(256, 3) dump_probe_kernel(int N, uint64_t n_chains, float* conf, double* lnW)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int gl = threadIdx.x & (G - 1);
    const uint32_t group = threadIdx.x / G, gpb = blockDim.x / G;
    float4* R4 = reinterpret_cast<float4*>(smem_raw + group_bytes(N, G, false) * group);
    for (int i = gl; i < N; i += G) R4[i] = make_float4((float)i, 0.5f * (float)i, -(float)i, 0.f);
    __syncwarp();
    for (uint64_t idx = (uint64_t)blockIdx.x * gpb + group; idx < n_chains; idx += (uint64_t)gridDim.x * gpb) {
        store_conf<G>(R4, conf + idx * (uint64_t)N * 3, N, N, gl);
        if (gl == 0 && lnW) lnW[idx] = (double)idx;
    }
}

// MSEQ: the per-step m sequence is requested (one shared-memory byte per step). The conformation dump needs no
// variant: the chain is in shared memory anyway and is stored once, after the last step, if p.out.conf is set.
// WELL: square-well model of DESIGN.md 3.6 (rosen_realspace_generate_model): contacts inside lambda sigma are counted
// per trial, the trial factors are the fixed-point Q[c], the choice is proportional to them, and the chain's result goes to
// a record (reduced afterwards with the largest lnW of the call as the shift) instead of the block partial.
template <int G, int P, bool DIGEST, bool MSEQ, bool WELL>
__global__ void __launch_bounds__(256, 3) realspace_kernel(const RealParams p)
{
    constexpr int T = 2 * P;                                 // trials per lane: t = T * gl + i, i = 0..T-1
    constexpr uint32_t kFull = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* ln_tab = reinterpret_cast<double*>(smem_raw);
    Partial* scratch = reinterpret_cast<Partial*>(smem_raw + 256 * sizeof(double));
    uint64_t* Qs = reinterpret_cast<uint64_t*>(smem_raw + 256 * sizeof(double) + 32 * sizeof(Partial));
    unsigned char* gbase_ptr = smem_raw + kFixedBytes;

    const int N = p.N, k = p.k, Np = n_pad(N);
    const int lane = threadIdx.x & 31;
    const int gl = lane & (G - 1);                         // lane within the group
    const int gshift = lane & ~(G - 1);                    // first lane of the group in the warp
    const uint32_t gmask = (G == 32) ? 0xffffffffu : ((1u << G) - 1u);
    const uint32_t below = (1u << gl) - 1u;
    const int group_in_block = threadIdx.x / G;
    float4* R4 = reinterpret_cast<float4*>(gbase_ptr + group_bytes(N, G, MSEQ) * group_in_block);   // one LDS.128 per monomer
    uint8_t* mbuf = reinterpret_cast<uint8_t*>(R4 + Np);

    for (int i = threadIdx.x; i < 256; i += blockDim.x) ln_tab[i] = i == 0 ? -CUDART_INF : log((double)i);
    if (threadIdx.x < 32) Qs[threadIdx.x] = p.Q[threadIdx.x];
    __syncthreads();
    // shared-window address of ln_tab kept in a register (opaque): the compiler otherwise re-derives it in every step
    uint32_t ln_addr = (uint32_t)__cvta_generic_to_shared(ln_tab);
    asm volatile("" : "+r"(ln_addr));

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
        const bool active = idx < p.n_chains;               // inactive groups of a warp with active ones compute and discard
        if (!__any_sync(kFull, active)) break;              // idx grows with it: this warp has no chain left in the virtual block
        const uint64_t chain = p.chain_offset + idx;
        const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);

        // R0
        for (int i = gl; i < Np; i += G) R4[i] = make_float4(kFar, kFar, kFar, 0.f);
        float hx = 0.f, hy = 0.f, hz = 0.f;
        double lnW = 0.0;
        bool alive = true;
        uint32_t steps = 0;
        uint64_t dg = 0xCBF29CE484222325ull;
        uint32_t selw[4] = {0, 0, 0, 0};
        uint32_t usel = 0;
        __syncwarp();

        for (int s = 1; s < N; ++s) {
            // selection word u_s = word s & 3 of block s >> 2: lane gl draws the blocks with (s >> 2) = gl (mod G), once per
            // 4 G steps, and the owner's word is broadcast (one Philox block per 4 steps and GROUP instead of per lane)
            if (s == 1 || (s & (4 * G - 1)) == 0)
                philox4x32_10(c_lo, c_hi, (uint32_t)(((s >> 2) & ~(G - 1)) + gl), 0u, p.key0, p.key1, selw);
            {   // word s & 3 without a dynamically indexed (local-memory) array
                const uint32_t lo = (s & 1) ? selw[1] : selw[0], hi = (s & 1) ? selw[3] : selw[2];
                usel = (s & 2) ? hi : lo;
                if constexpr (G > 1) usel = __shfl_sync(kFull, usel, gshift + ((s >> 2) & (G - 1)));
            }

            // ---- R1: this lane's trials (P Philox blocks = 2P consecutive trials)
            float tx[T], ty[T], tz[T];
            float near2[T];                                  // smallest spec'd d2 to an earlier monomer so far (-1: trial index >= k)
            uint32_t nwell[T];                               // WELL: earlier monomers with d2 < well2
#pragma unroll
            for (int pp = 0; pp < P; ++pp) {
                const uint32_t bi = (uint32_t)(P * gl + pp);
                uint32_t w[4];
                philox4x32_10(c_lo, c_hi, (uint32_t)s, 1u + bi, p.key0, p.key1, w);
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    float ux, uy, uz;
                    direction(w[2 * e], w[2 * e + 1], ux, uy, uz);
                    tx[2 * pp + e] = __fmaf_rn(p.b, ux, hx);
                    ty[2 * pp + e] = __fmaf_rn(p.b, uy, hy);
                    tz[2 * pp + e] = __fmaf_rn(p.b, uz, hz);
                    near2[2 * pp + e] = (int)(2u * bi + e) < k ? CUDART_MAX_NORMAL_F : -1.0f;
                    nwell[2 * pp + e] = 0u;
                }
            }

            // ---- R2: monomers j <= s-2 (slots 0..s-2; r_{s-1} itself is stored at the end of this step), 32 per pass:
            // mark those within the conservative radius of r_{s-1}, then test the trials against the marked ones
            // (overlap is an OR over monomers: order and batching are irrelevant)
            auto test_marked = [&](uint32_t mask, const float4* pb) {
                while (mask) {
                    const uint32_t bpos = bfind(mask);
                    mask ^= 1u << bpos;
                    const float4 rj = pb[bpos];
#pragma unroll
                    for (int i = 0; i < T; ++i) {
                        const float dx = __fsub_rn(rj.x, tx[i]), dy = __fsub_rn(rj.y, ty[i]), dz = __fsub_rn(rj.z, tz[i]);
                        const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                        near2[i] = fminf(near2[i], d2);      // overlap iff some d2 < sigma2 iff the smallest is
                        if (WELL) nwell[i] += d2 < p.well2 ? 1u : 0u;
                    }
                }
            };
            {
                const int cnt = s - 1;
                int j0 = 0;
                if constexpr (G == 32) {
                    // two passes per iteration while two remain: independent loads and distance chains, half the loop overhead
                    for (; j0 + 32 < cnt; j0 += 64) {
                        const float4* pb = R4 + j0;
                        const uint32_t m0 = candidate_bits<G>(pb, 32, gl, gshift, gmask, hx, hy, hz, p.prefilter2);
                        const uint32_t m1 = candidate_bits<G>(pb + 32, 32, gl, gshift, gmask, hx, hy, hz, p.prefilter2);
                        test_marked(m0, pb);
                        test_marked(m1, pb + 32);
                    }
                }
                for (; j0 < cnt; j0 += 32)
                    test_marked(candidate_bits<G>(R4 + j0, cnt - j0, gl, gshift, gmask, hx, hy, hz, p.prefilter2), R4 + j0);
            }

            // ---- m_s and the number of free trials of lower lanes (trial order = lane order, then i)
            uint32_t f = 0;
#pragma unroll
            for (int i = 0; i < T; ++i) f |= near2[i] < p.sigma2 ? 0u : 1u << i;
            const uint32_t c = __popc(f);
            uint32_t m, excl;
            if constexpr (G == 1) {
                m = c; excl = 0;
            } else if constexpr (G <= 4) {
                uint32_t V = c << (8 * gl);                  // one byte per lane (c <= 8)
#pragma unroll
                for (int d = 1; d < G; d <<= 1) V |= __shfl_xor_sync(kFull, V, d);
                const uint32_t cum = V * 0x01010101u;        // byte j = c_0 + ... + c_j (no carries: total <= 32)
                m = cum >> 24;
                excl = ((cum << 8) >> (8 * gl)) & 0xFFu;
            } else {
                m = 0; excl = 0;
#pragma unroll
                for (int i = 0; i < T; ++i) {
                    const uint32_t B = (__ballot_sync(kFull, (f >> i) & 1u) >> gshift) & gmask;
                    m += __popc(B); excl += __popc(B & below);
                }
            }

            // ---- R3
            steps += alive ? 1u : 0u;
            if (MSEQ) { if (gl == 0) mbuf[s - 1] = alive ? (uint8_t)m : (uint8_t)0; }

            // ---- R4
            bool hit;
            int li;
            if constexpr (!WELL) {
                if constexpr (G >= 16) { double lm; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(lm) : "r"(ln_addr + 8u * m)); lnW += lm; }
                else lnW += ln_tab[m];                       // (measured: the register copy helps G = 32 by 1.2 %, costs G = 4 1.5 %)
                // the sel-th free trial; it is this lane's if excl <= sel < excl + c, namely the (sel - excl)-th set bit of f
                const uint32_t sel = __umulhi(usel, m);
                const uint32_t rk = sel - excl;
                hit = rk < c;
                uint32_t g2 = f;
#pragma unroll
                for (int i = 0; i < T - 1; ++i) g2 = (rk > (uint32_t)i) ? (g2 & (g2 - 1u)) : g2;
                li = __ffs(g2) - 1;
            } else {
                // Boltzmann-weighted choice: integer factors, so the group's prefix sums are exact
                uint64_t lw[T], Ls = 0;
#pragma unroll
                for (int i = 0; i < T; ++i) { lw[i] = ((f >> i) & 1u) ? Qs[min(nwell[i], 31u)] : 0ull; Ls += lw[i]; }
                uint64_t inc = Ls;
#pragma unroll
                for (int d = 1; d < G; d <<= 1) {
                    const uint64_t v = __shfl_up_sync(kFull, (unsigned long long)inc, d, G);
                    if (gl >= d) inc += v;
                }
                const uint64_t Wt = G > 1 ? (uint64_t)__shfl_sync(kFull, (unsigned long long)inc, gshift + G - 1) : inc;
                lnW += log((double)Wt * 0x1p-16);            // log(0) = -inf for a dead end
                const uint64_t target = (Wt >> 32) * (uint64_t)usel + (((Wt & 0xFFFFFFFFull) * (uint64_t)usel) >> 32);
                uint64_t cum = inc - Ls;
                hit = Wt != 0ull && target >= cum && target < inc;
                li = T - 1;
                bool found = false;
#pragma unroll
                for (int i = 0; i < T; ++i) {
                    cum += lw[i];
                    if (!found && cum > target) { found = true; li = i; }
                }
            }
            float px = tx[0], py = ty[0], pz = tz[0];
#pragma unroll
            for (int i = 1; i < T; ++i)
                if (li == i) { px = tx[i]; py = ty[i]; pz = tz[i]; }
            uint32_t tsel = (uint32_t)(T * gl + li);
            if constexpr (G > 1) {
                const uint32_t hb = (__ballot_sync(kFull, hit) >> gshift) & gmask;
                const int src = gshift + (hb ? __ffs(hb) - 1 : 0);
                px = __shfl_sync(kFull, px, src); py = __shfl_sync(kFull, py, src); pz = __shfl_sync(kFull, pz, src);
                if (DIGEST) tsel = __shfl_sync(kFull, tsel, src);
            }
            if (DIGEST) { if (alive) dg = digest_fold(dg, m, m ? tsel : 0xFFu); }
            if (gl == 0) R4[s - 1] = make_float4(hx, hy, hz, 0.f);      // r_{s-1} becomes scannable from step s+1 on
            alive = alive && (m != 0u);
            if (m != 0u) { hx = px; hy = py; hz = pz; }
            __syncwarp();
        }
        if (gl == 0) R4[N - 1] = make_float4(hx, hy, hz, 0.f);
        __syncwarp();

        // ---- R5: fp64 sums over the finished chain, the group's lanes in parallel, then a butterfly (every lane
        // of the group ends with the same bits: a + b == b + a)
        double Sx = 0.0, Sy = 0.0, Sz = 0.0, S2 = 0.0;
        for (int i = gl; i < N; i += G) {
            const float4 r = R4[i];
            const double x = (double)r.x, y = (double)r.y, z = (double)r.z;
            Sx += x; Sy += y; Sz += z; S2 += x * x + y * y + z * z;
        }
#pragma unroll
        for (int d = 1; d < G; d <<= 1) {
            Sx += __shfl_xor_sync(kFull, Sx, d); Sy += __shfl_xor_sync(kFull, Sy, d);
            Sz += __shfl_xor_sync(kFull, Sz, d); S2 += __shfl_xor_sync(kFull, S2, d);
        }
        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            ree2 = (double)hx * (double)hx + (double)hy * (double)hy + (double)hz * (double)hz;
            const double inv = 1.0 / (double)N;
            const double cx = Sx * inv, cy = Sy * inv, cz = Sz * inv;
            rg2 = S2 * inv - (cx * cx + cy * cy + cz * cz);
        }
        const double wgt = (alive && !WELL) ? exp(lnW - p.ln_shift) : 0.0;
        if (WELL) {
            if (active && gl == 0) {
                ChainRecord rc;
                rc.lnW = alive ? lnW : -CUDART_INF; rc.ree2 = ree2; rc.rg2 = rg2;
                rc.steps = steps; rc.alive = alive ? 1u : 0u; rc.digest = dg;
                p.rec[idx] = rc;
            }
        } else if (active && gl == 0) {
            acc.sum_w += wgt; acc.sum_w_ree2 += wgt * ree2; acc.sum_w_rg2 += wgt * rg2; acc.sum_w2 += wgt * wgt;
            acc.n_dead += alive ? 0u : 1u; acc.n_steps += steps;
            if (DIGEST) { acc.digest_xor ^= dg; acc.digest_sum += dg; }
            if (p.out.lnW) p.out.lnW[idx] = lnW;
            if (p.out.alive) p.out.alive[idx] = alive ? 1 : 0;
            if (p.out.ree2) p.out.ree2[idx] = ree2;
            if (p.out.rg2) p.out.rg2[idx] = rg2;
            if (DIGEST && p.out.digest) p.out.digest[idx] = dg;
        }
        // ---- D1
        if (p.out.conf != nullptr && active)
            store_conf<G>(R4, reinterpret_cast<float*>(p.out.conf) + idx * (uint64_t)N * 3, N, alive ? N : (int)steps, gl);
        if (MSEQ && active) {
            uint8_t* mr = p.out.m_seq + idx * (uint64_t)(N - 1);
            for (int e = gl; e < N - 1; e += G) mr[e] = mbuf[e];
        }
        __syncwarp();
    }

    if (WELL) __syncthreads();      // the sums are formed from the records afterwards; the ticket still needs the barrier
    else block_reduce_store(acc, scratch, p.partials + vb);
    if (p.done != nullptr) {        // every thread's stores of this virtual block are visible system-wide before the flag is
        __threadfence_system();
        __syncthreads();
        if (threadIdx.x == 0) { *reinterpret_cast<volatile uint32_t*>(p.done + vb) = 1u; __threadfence_system(); }
    }
    }
}

// threads per block: a function of (N, G) only -- it fixes the reduction tree, so it must not depend on the output variant
int block_threads(int N, int G)
{
    const size_t fixed = kFixedBytes;
    const size_t gsz = group_bytes(N, G, true);
    int threads = 256;
    while (threads > 32 && fixed + gsz * (threads / G) > (size_t)(74 * 1024 + 512)) threads >>= 1;   // three blocks per SM
    return threads;
}

template <int G, int P, bool DIGEST, bool MSEQ, bool WELL>
int launch_one(const RealParams& p, cudaStream_t stream, int* grid_out)
{
    int dev = 0, n_sm = 0, smem_max = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t fixed = kFixedBytes;
    const int threads = block_threads(p.N, G);
    const size_t smem = fixed + group_bytes(p.N, G, MSEQ) * (threads / G);
    if (smem > (size_t)smem_max) return -2;
    auto kern = realspace_kernel<G, P, DIGEST, MSEQ, WELL>;
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
    const bool mseq = p.out.m_seq != nullptr;
    if (p.rec != nullptr)          // square-well model: the record always carries the digest
        return mseq ? launch_one<G, P, true, true, true>(p, stream, grid_out) : launch_one<G, P, true, false, true>(p, stream, grid_out);
    if (mseq) return digest ? launch_one<G, P, true, true, false>(p, stream, grid_out) : launch_one<G, P, false, true, false>(p, stream, grid_out);
    return digest ? launch_one<G, P, true, false, false>(p, stream, grid_out) : launch_one<G, P, false, false, false>(p, stream, grid_out);
}

// direction map alone (test entry rosen_direction_eval): out[3 i ..] = direction(wz[i], wphi[i])
__global__ void direction_eval_kernel(const uint32_t* __restrict__ wz, const uint32_t* __restrict__ wphi, uint64_t n,
                                      float* __restrict__ out)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        float ux, uy, uz;
        direction(wz[i], wphi[i], ux, uy, uz);
        out[3 * i] = ux; out[3 * i + 1] = uy; out[3 * i + 2] = uz;
    }
}

}  // namespace

int launch_direction_eval(const uint32_t* wz, const uint32_t* wphi, uint64_t n, float* out, cudaStream_t stream)
{
    const uint64_t blocks = (n + 255) / 256;
    direction_eval_kernel<<<(int)(blocks < 4096 ? blocks : 4096), 256, 0, stream>>>(wz, wphi, n, out);
    return cudaGetLastError() == cudaSuccess ? 1 : -3;
}

int launch_dump_probe(int N, uint64_t n_chains, float* conf, double* lnW, cudaStream_t stream)
{
    constexpr int G = 32;                                    // the geometry of BASELINE config 5 (k = 64: one warp per chain)
    int dev = 0, n_sm = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    const int threads = block_threads(N, G);
    const size_t smem = group_bytes(N, G, false) * (threads / G);
    auto kern = dump_probe_kernel<G>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -3;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) return -3;
    const uint64_t want = (n_chains + threads / G - 1) / (threads / G), cap = (uint64_t)n_sm * per_sm;
    kern<<<(int)(want < cap ? want : cap), threads, smem, stream>>>(N, n_chains, conf, lnW);
    return cudaGetLastError() == cudaSuccess ? 1 : -3;
}

int launch_realspace(const RealParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out)
{
    int blocks = (p.k + 1) / 2;   // Philox blocks (trial pairs) per step
    // Long chains: a warp holds 32/G chains of group_bytes(N) each; widen the group (idle lanes own trials >= k)
    // until one warp's chains fit 24 KB, so that a block of >= 4 warps fits shared memory (N = 2048: one chain per warp, 2 warps per block).
    {
        const size_t gsz = (size_t)n_pad(p.N) * 17;
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
