// lattice_hash.cu -- cubic-lattice Rosenbluth generation for LONG chains (193 <= N <= 16383), the range of the
// paper's "global-memory version" (Table 1; Fig. 2b, :296) and of its longest shared-memory
// rows (N = 1024, 2048, :280-281). Same steps L0-L5 and the same decisions as lattice.cu, but
// the occupancy scan of Alg. 1 lines 13-17, which costs O(s) per step, is replaced by an
// exact per-chain hash map of occupied sites in global memory: O(N) per chain instead of O(N^2)
// ("a per-chain hash set would make it ~5 probes/step").
//
// Layout. One thread grows one chain. Space is cut into 4 x 4 x 4 cubes; the chain's table maps a
// cube to the 64-bit occupancy bitmap of its sites. An entry is 16 bytes:
//   .x  bits 0..38   cube key (cx+2^12) | (cy+2^12) << 13 | (cz+2^12) << 26, c = coordinate >> 2 (floor)
//       bits 39..63  the thread's chain generation (1, 2, ...): an entry whose generation differs from the current
//                    chain's is EMPTY, so tables are never cleared between chains, nor between calls of the same
//                    table layout: the counter is kept in the workspace (one memset per allocation or layout change)
//   .y  bit (x&3) | (y&3) << 2 | (z&3) << 4 set = site occupied
// Tables are open-addressed (Fibonacci hash of the cube key reduced by a multiply-high, linear probing, no deletions)
// with N+1 entries (rounded up to even): a chain of N monomers touches at most N cubes, so a probe always ends at an
// empty entry; on average a chain touches about N/6 cubes, so probes longer than one entry are rare.
// The growth point's own cube lives in registers (bitmap + entry index); of the six neighbour sites only those
// across a cube face need memory: at most three look-ups per step, 1.5 on average, against five for a per-site set,
// and the insert is a 16-byte store to an entry that is already known.
//
// Scheduling. Chains of this length die often (attrition 20 % at N = 1024, 93 % at N = 10000) and run for very
// different times, so lanes draw chain indices from a global ticket one by one and every warp iteration is one
// growth step of each lane's current chain -- no lane waits for its neighbours' chains. Because that order is
// timing dependent, the kernel only writes one fixed-size record per chain; the ensemble sums are formed afterwards
// by reduce_records_kernel over virtual blocks in a fixed order (deterministic, grid independent, no float
// atomics), which also writes the optional per-chain outputs, coalesced.
//
// Roofline: issue slots (ncu: 60 % issue-active, 28 % of DRAM peak; the first per-site version was DRAM bound), DESIGN.md 5.5 / 6.
#include <cstdlib>
#include <math_constants.h>
#include "common.cuh"
#include "philox.cuh"
#include "reduce.cuh"

namespace rosen {

namespace {

constexpr int      kCubeField = 13;
constexpr uint64_t kCubeBias = 1ull << (kCubeField - 1);
constexpr uint64_t kOriginCube = kCubeBias | (kCubeBias << kCubeField) | (kCubeBias << (2 * kCubeField));
constexpr int      kGenShift = 3 * kCubeField;                       // 39
constexpr uint32_t kGenMax = (1u << (64 - kGenShift)) - 1u;

__device__ __forceinline__ uint64_t digest_fold(uint64_t h, uint32_t m, uint32_t choice)
{
    return (h ^ (uint64_t)(m | (choice << 8))) * 0x100000001B3ull;
}

// home entry of a cube. The 2 x 2 x 2 block of cubes it belongs to (cube coordinates >> 1) is hashed to a group of 8
// consecutive entries = one 128-byte line (Fibonacci hash, range-reduced by a multiply-high), and the low coordinate bits
// pick the entry inside the line: a walk's consecutive cubes are neighbours in space, so they share lines instead of
// touching one random 32-byte sector each (DRAM bytes per step: section 12). Probing stays linear over the whole table.
__device__ __forceinline__ uint32_t slot_of_local(uint64_t cube, uint32_t entries)
{
    constexpr uint64_t kLow = 1ull | (1ull << kCubeField) | (1ull << (2 * kCubeField));
    const uint32_t low = (uint32_t)(cube & 1ull) | ((uint32_t)(cube >> (kCubeField - 1)) & 2u) | ((uint32_t)(cube >> (2 * kCubeField - 2)) & 4u);
    return __umulhi((uint32_t)(((cube & ~kLow) * 0x9E3779B97F4A7C15ull) >> 32), entries >> 3) * 8u + low;
}

// Very long chains fill whole lines with neighbouring cubes and then probe through them (N = 10000: 104 -> 124 ms with the
// line-local hash), so from kLocalHashMaxN on every cube is hashed on its own.
constexpr int kLocalHashMaxN = 4096;
__device__ __forceinline__ uint32_t slot_of(uint64_t cube, uint32_t entries, bool local)
{
    return local ? slot_of_local(cube, entries) : __umulhi((uint32_t)((cube * 0x9E3779B97F4A7C15ull) >> 32), entries);
}

// three-way select by axis
template <typename T> __device__ __forceinline__ T pick(uint32_t a, T v0, T v1, T v2) { return a == 0u ? v0 : (a == 1u ? v1 : v2); }

template <bool TRAJ, bool DIGEST>
__global__ void __launch_bounds__(256, 3) lattice_hash_kernel(const HashParams p)
{
    __shared__ double ln_m[8];
    __shared__ uint8_t nth_free[64 * 8];    // [free-direction mask][sel] -> the sel-th free direction, order +x,-x,+y,-y,+z,-z
    if (threadIdx.x < 8) ln_m[threadIdx.x] = threadIdx.x == 0 ? -CUDART_INF : log((double)threadIdx.x);
    for (uint32_t i = threadIdx.x; i < 64u * 8u; i += blockDim.x) {
        uint32_t fr = i >> 3;
        for (uint32_t k = 0; k < (i & 7u); ++k) fr &= fr - 1u;
        nth_free[i] = (uint8_t)(fr ? __ffs((int)fr) - 1 : 0);
    }
    __syncthreads();

    const int N = p.N;
    const uint32_t entries = p.entries;
    const bool local_hash = N <= kLocalHashMaxN;
    ulonglong2* table = reinterpret_cast<ulonglong2*>(p.tables) + ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * entries;
    const uint64_t gthread = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t gen = p.gen_store[gthread];    // generations continue across calls: entries of earlier calls stay "empty" without a memset
    uint32_t t = 0;                         // warp iteration counter (uniform): Philox blocks are drawn when t & 3 == 0

    // per-lane state of the chain being grown; s == 0: the lane needs a new chain
    uint64_t idx = 0, tag = 0, dg = 0;
    uint64_t cube = 0, bits = 0;            // the growth point's cube: key and occupancy bitmap (register copy of its entry)
    uint32_t slot = 0, l = 0;               // its entry index; local site index of the growth point inside it
    uint32_t c_lo = 0, c_hi = 0, w[4] = {0u, 0u, 0u, 0u}, wn[4] = {0u, 0u, 0u, 0u};
    int s = 0, x = 0, y = 0, z = 0, sx = 0, sy = 0, sz = 0;
    long long s2 = 0;
    double lnW = 0.0;
    uint8_t* mrow = nullptr;
    int32_t* crow = nullptr;

    // One iteration = one growth step of every lane's current chain. A lane whose chain ended (full length or dead
    // end) writes its record and draws the next chain in the same iteration, so no lane idles while its neighbours'
    // chains are still growing.
    for (;;) {
        if (s == 0) {
            // ---- draw the next chain (timing dependent; results are not: a record is a function of the chain id)
            idx = atomicAdd(p.ticket, 1ull);
            if (idx >= p.n_chains) { p.gen_store[gthread] = gen; break; }
            const uint64_t chain = p.chain_offset + idx;
            c_lo = (uint32_t)chain; c_hi = (uint32_t)(chain >> 32);
            if (++gen > kGenMax) {     // generation counter wrapped: clear the table once and start over
                for (uint32_t i = 0; i < entries; ++i) table[i] = make_ulonglong2(0ull, 0ull);
                gen = 1u;
            }
            tag = (uint64_t)gen << kGenShift;
            // ---- L0: r_0 = origin; every entry is empty for a new generation, so the origin's cube takes its home slot
            cube = kOriginCube; bits = 1ull; l = 0u;
            slot = slot_of(cube, entries, local_hash);
            table[slot] = make_ulonglong2(cube | tag, bits);
            x = y = z = sx = sy = sz = 0; s2 = 0; lnW = 0.0; s = 1;
            dg = 0xCBF29CE484222325ull;
            philox4x32_10(c_lo, c_hi, 0u, 0u, p.key0, p.key1, w);             // L1, block of steps 1..3
            if (TRAJ) {
                mrow = p.out.m_seq ? p.out.m_seq + idx * (uint64_t)(N - 1) : nullptr;
                crow = p.out.conf ? reinterpret_cast<int32_t*>(p.out.conf) + idx * (uint64_t)N * 3 : nullptr;
                if (crow) { crow[0] = 0; crow[1] = 0; crow[2] = 0; }
            }
        }
        // ---- L1. Lanes are at different steps of their chains; drawing a block whenever some lane enters a new group
        // of four steps would run the Philox rounds in almost every iteration for a few lanes. Instead every fourth
        // iteration ALL lanes draw the block of the next group they will enter, (s+3) >> 2 (the current group if
        // s & 3 == 0), into wn, and a lane switches to it on entering that group -- which happens within four steps.
        if ((t & 3u) == 0u) philox4x32_10(c_lo, c_hi, (uint32_t)(s + 3) >> 2, 0u, p.key0, p.key1, wn);
        ++t;
        if ((s & 3) == 0) { w[0] = wn[0]; w[1] = wn[1]; w[2] = wn[2]; w[3] = wn[3]; }

        // ---- L2. Per axis at most one neighbour site lies across a cube face (local coordinate 0 or 3): fetch that
        // cube's bitmap (all first probes in flight together); the other neighbours are bits of the register bitmap.
        uint64_t nkey[3], nbits[3];
        uint32_t nslot[3], nl[3];
        ulonglong2 first[3];
        bool need[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const uint32_t la = (l >> (2 * a)) & 3u;
            const bool up = la == 3u;
            need[a] = up || la == 0u;
            nkey[a] = up ? cube + (1ull << (kCubeField * a)) : cube - (1ull << (kCubeField * a));
            nl[a] = (up ? l - (3u << (2 * a)) : l + (3u << (2 * a))) & 63u;
            // no face on this axis: probe the growth point's own entry instead (cached, never a match for nkey, never
            // empty) so that the load needs no branch; its result is not used
            nslot[a] = need[a] ? slot_of(nkey[a], entries, local_hash) : slot;
            first[a] = table[nslot[a]];
        }
        uint32_t pend = 0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const bool hit = first[a].x == (nkey[a] | tag);
            nbits[a] = hit ? first[a].y : 0ull;
            pend |= (need[a] && (uint32_t)(first[a].x >> kGenShift) == gen && !hit) ? 1u << a : 0u;
        }
        while (pend) {
            // home entry taken by another cube of this chain (tables are ~1/6 full at most on average): one shared
            // probe loop for whichever axes need it
            const uint32_t a = (uint32_t)__ffs((int)pend) - 1u;
            pend &= pend - 1u;
            const uint64_t want = pick(a, nkey[0], nkey[1], nkey[2]) | tag;
            uint32_t sl = pick(a, nslot[0], nslot[1], nslot[2]);
            uint64_t nb = 0ull;
            for (;;) {
                sl = sl + 1u == entries ? 0u : sl + 1u;
                const ulonglong2 e = table[sl];
                if ((uint32_t)(e.x >> kGenShift) != gen) break;                    // empty: cube not visited yet; sl = where it would go
                if (e.x == want) { nb = e.y; break; }
            }
            if (a == 0u) { nslot[0] = sl; nbits[0] = nb; }
            if (a == 1u) { nslot[1] = sl; nbits[1] = nb; }
            if (a == 2u) { nslot[2] = sl; nbits[2] = nb; }
        }
        uint32_t occ = 0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const uint32_t la = (l >> (2 * a)) & 3u;
            const uint32_t in_up = (uint32_t)(bits >> ((l + (1u << (2 * a))) & 63u)) & 1u;
            const uint32_t in_dn = (uint32_t)(bits >> ((l - (1u << (2 * a))) & 63u)) & 1u;
            const uint32_t out = (uint32_t)(nbits[a] >> nl[a]) & 1u;
            occ |= (la == 3u ? out : in_up) << (2 * a);             // +axis
            occ |= (la == 0u ? out : in_dn) << (2 * a + 1);         // -axis
        }
        const uint32_t m = 6u - (uint32_t)__popc(occ);
        if (TRAJ && mrow) mrow[s - 1] = (uint8_t)m;

        bool done;
        if (m == 0u) {
            // ---- L3: dead end (W = 0, chain kept; reading A6)
            if (DIGEST) dg = digest_fold(dg, 0u, 0xFFu);
            done = true;
        } else {
            lnW += ln_m[m];
            // ---- L4
            const uint32_t u = (s & 2) ? ((s & 1) ? w[3] : w[2]) : ((s & 1) ? w[1] : w[0]);
            const uint32_t sel = __umulhi(u, m);
            const uint32_t d = nth_free[((~occ & 63u) << 3) + sel];
            if (DIGEST) dg = digest_fold(dg, m, d);
            const uint32_t a = d >> 1;
            const bool up = (d & 1u) == 0u;
            const uint32_t la = (l >> (2u * a)) & 3u;
            const bool cross = up ? la == 3u : la == 0u;      // across a cube face: that cube's entry becomes the register copy
            const uint32_t l_in = up ? l + (1u << (2u * a)) : l - (1u << (2u * a));
            cube = cross ? pick(a, nkey[0], nkey[1], nkey[2]) : cube;
            slot = cross ? pick(a, nslot[0], nslot[1], nslot[2]) : slot;
            bits = cross ? pick(a, nbits[0], nbits[1], nbits[2]) : bits;
            l = cross ? pick(a, nl[0], nl[1], nl[2]) : l_in;
            bits |= 1ull << l;
            table[slot] = make_ulonglong2(cube | tag, bits);              // insert r_s (write-through; L2 absorbs repeats)
            const int sg = up ? 1 : -1;
            x += a == 0u ? sg : 0; y += a == 1u ? sg : 0; z += a == 2u ? sg : 0;
            if (TRAJ && crow) { crow[3 * s + 0] = x; crow[3 * s + 1] = y; crow[3 * s + 2] = z; }
            // ---- L5
            sx += x; sy += y; sz += z; s2 += (long long)(x * x + y * y + z * z);
            ++s;
            done = s == N;
        }

        if (done) {
            const bool alive = m != 0u;
            if (TRAJ && !alive) {      // zero-fill from the death step on (reading A13); m_seq[s-1] = 0 is already there
                if (mrow) for (int q = s; q < N - 1; ++q) mrow[q] = 0;
                if (crow) for (int q = 3 * s; q < 3 * N; ++q) crow[q] = 0;
            }
            ChainRecord r;
            r.lnW = alive ? lnW : -CUDART_INF;
            r.ree2 = 0.0; r.rg2 = 0.0;
            if (alive) {
                r.ree2 = (double)((long long)x * x + (long long)y * y + (long long)z * z);
                const long long num = (long long)N * s2 - ((long long)sx * sx + (long long)sy * sy + (long long)sz * sz);
                r.rg2 = (double)num / ((double)N * (double)N);
            }
            r.steps = alive ? (uint32_t)(N - 1) : (uint32_t)s;     // attempted steps
            r.alive = alive ? 1u : 0u;
            r.digest = DIGEST ? dg : 0ull;
            p.rec[idx] = r;
            s = 0;
        }
    }
}

// Long chains proper (lattice N > 512, real space N > 2048, reading A18): the shift L of the weights is the
// largest lnW of the call, found by two max passes over the records (max is exact and order independent) and kept
// in device memory for the sums and for the summary. lmax[0..n_vblocks) = block maxima, lmax[kMaxPartials] = L.
__global__ void __launch_bounds__(256) records_max_kernel(const ChainRecord* __restrict__ rec, uint64_t n_chains, uint32_t chunk,
                                                          double* lmax)
{
    __shared__ double sm[8];
    double v = -CUDART_INF;
    for (uint32_t it = 0; it < chunk / 256u; ++it) {
        const uint64_t idx = (uint64_t)blockIdx.x * chunk + (uint64_t)it * 256u + threadIdx.x;
        if (idx >= n_chains) break;
        if ((rec[idx].alive & 1u) != 0u) v = fmax(v, rec[idx].lnW);
    }
    for (int d = 16; d >= 1; d >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, d));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) v = fmax(v, sm[w]);
        lmax[blockIdx.x] = v;
    }
}

__global__ void __launch_bounds__(256) records_max_final_kernel(double* lmax, uint32_t n_vblocks)
{
    __shared__ double sm[8];
    double v = -CUDART_INF;
    for (uint32_t i = threadIdx.x; i < n_vblocks; i += 256u) v = fmax(v, lmax[i]);
    for (int d = 16; d >= 1; d >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, d));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) v = fmax(v, sm[w]);
        lmax[kMaxPartials] = v == -CUDART_INF ? 0.0 : v;       // no chain alive: L = 0, all weights 0
    }
}

// E1, first pass, for kernels that write per-chain records: virtual block v sums the chains [v*chunk, (v+1)*chunk)
// with the thread mapping and tree of the generation kernels (thread t takes v*chunk + it*256 + t, it ascending).
// ln_shift_dev != nullptr: the shift is read from device memory (long chains), else ln_shift is used.
__global__ void __launch_bounds__(256) reduce_records_kernel(const ChainRecord* __restrict__ rec, uint64_t n_chains, uint32_t chunk,
                                                             double ln_shift, const double* ln_shift_dev, DevOutputs out, Partial* partials)
{
    __shared__ Partial scratch[8];
    const uint32_t vb = blockIdx.x;
    if (ln_shift_dev) ln_shift = *ln_shift_dev;
    Partial acc = partial_zero();
    for (uint32_t it = 0; it < chunk / 256u; ++it) {
        const uint64_t idx = (uint64_t)vb * chunk + (uint64_t)it * 256u + threadIdx.x;
        if (idx >= n_chains) break;
        const ChainRecord r = rec[idx];
        const bool alive = (r.alive & 1u) != 0u;                       // bit 1 (PERM): tour stopped at max_nodes, reported as 2
        const double wgt = alive ? exp(r.lnW - ln_shift) : 0.0;
        acc.sum_w += wgt; acc.sum_w_ree2 += wgt * r.ree2; acc.sum_w_rg2 += wgt * r.rg2; acc.sum_w2 += wgt * wgt;
        acc.n_dead += alive ? 0u : 1u; acc.n_steps += r.steps;
        if (out.digest) { acc.digest_xor ^= r.digest; acc.digest_sum += r.digest; out.digest[idx] = r.digest; }
        if (out.lnW) out.lnW[idx] = r.lnW;
        if (out.alive) out.alive[idx] = (r.alive & 2u) ? 2 : (alive ? 1 : 0);
        if (out.ree2) out.ree2[idx] = r.ree2;
        if (out.rg2) out.rg2[idx] = r.rg2;
    }
    block_reduce_store(acc, scratch, partials + vb);
}

}  // namespace

uint32_t hash_entries(int32_t N)
{
    return ((uint32_t)N + 8u) & ~7u;                   // a multiple of 8 (whole 128-byte lines) and >= N + 1 > cubes one chain can touch
}

uint32_t lattice_hash_gen_max() { return kGenMax; }

int hash_max_threads(int* threads_out, int blocks_per_sm_cap)
{
    int dev = 0, n_sm = 0, per_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    // the traj variant has the larger register footprint: size the tables for the plain one, which every launch may use
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lattice_hash_kernel<false, false>, 256, 0) != cudaSuccess || per_sm < 1) return -3;
    if (blocks_per_sm_cap >= 1 && blocks_per_sm_cap < per_sm) per_sm = blocks_per_sm_cap;
    *threads_out = n_sm * per_sm * 256;
    return 0;
}

int launch_lattice_hash(const HashParams& p, int n_threads, cudaStream_t stream, const char** kernel_name)
{
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    const int grid = n_threads / 256;
    const bool digest = p.out.digest != nullptr;
    if (traj) {
        if (digest) { *kernel_name = "lattice_hash_kernel<digest,traj>"; lattice_hash_kernel<true, true><<<grid, 256, 0, stream>>>(p); }
        else        { *kernel_name = "lattice_hash_kernel<traj>";        lattice_hash_kernel<true, false><<<grid, 256, 0, stream>>>(p); }
    } else {
        if (digest) { *kernel_name = "lattice_hash_kernel<digest>";      lattice_hash_kernel<false, true><<<grid, 256, 0, stream>>>(p); }
        else        { *kernel_name = "lattice_hash_kernel";              lattice_hash_kernel<false, false><<<grid, 256, 0, stream>>>(p); }
    }
    if (cudaGetLastError() != cudaSuccess) return -3;
    const int rc = launch_reduce_records(p.rec, p.n_chains, p.chunk, p.n_vblocks, p.ln_shift, p.lmax, p.out, p.partials, stream);
    return rc < 0 ? rc : 1 + rc;
}

int launch_reduce_records(const ChainRecord* rec, uint64_t n_chains, uint32_t chunk, uint32_t n_vblocks, double ln_shift,
                          double* lmax, const DevOutputs& out, Partial* partials, cudaStream_t stream)
{
    int launches = 1;
    if (lmax) {
        records_max_kernel<<<n_vblocks, 256, 0, stream>>>(rec, n_chains, chunk, lmax);
        records_max_final_kernel<<<1, 256, 0, stream>>>(lmax, n_vblocks);
        launches = 3;
    }
    reduce_records_kernel<<<n_vblocks, 256, 0, stream>>>(rec, n_chains, chunk, ln_shift, lmax ? lmax + kMaxPartials : nullptr, out, partials);
    return cudaGetLastError() == cudaSuccess ? launches : -3;
}

}  // namespace rosen
