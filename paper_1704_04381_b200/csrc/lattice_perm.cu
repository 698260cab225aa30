// lattice_perm.cu -- PERM, the pruned-enriched Rosenbluth method, on the cubic lattice (DESIGN.md 3.7,
// readings A22-A24). The paper only names PERM as the topic of its unavailable supplement; the
// algorithm is Grassberger's (Phys. Rev. E 56, 3682 (1997)), depth-first, with caller-given thresholds.
//
// One thread runs one tour at a time and draws the next tour from a global ticket when its tour ends (tour sizes vary by
// orders of magnitude), inside the same flat loop in which the other lanes of its warp go on with theirs. The recursion of DESIGN.md 3.7 is an explicit stack: an enrichment pushes the second copy
// (length, lnW); the chain prefix it continues from is still in place when it is popped, because deeper levels only
// overwrite later monomers. The chain is one packed key per monomer (3 x 10-bit fields, bias 512; 2 <= N <= 512) in shared
// memory, laid out [monomer][thread]; the free-neighbour count is the scan of Alg. 1 over the monomers of the right
// parity (the lattice is bipartite: DESIGN.md 5.1). Every tour leaves one record; reduce_records_kernel forms the
// deterministic sums with the largest ln S of the call as the shift.
#include <math_constants.h>
#include "common.cuh"
#include "philox.cuh"

namespace rosen {

namespace {

constexpr int kField = 10, kBias = 512;
constexpr uint32_t kFieldMask = (1u << kField) - 1u;
constexpr int kMaxDepth = 512;

__device__ __forceinline__ uint64_t fold(uint64_t h, uint32_t m, uint32_t choice)
{
    return (h ^ (uint64_t)(m | (choice << 8))) * 0x100000001B3ull;
}

// prefix sums of the chain a stacked copy continues from (observables are formed from running sums, not by a pass over the
// chain at every leaf: a leaf then costs as much as any other node, which the lock-step loop below needs)
struct Sums { int sx, sy, sz, s2; };     // |coordinate| <= 511: s2 <= 512 x 3 x 511^2 < 2^31

__global__ void __launch_bounds__(128) lattice_perm_kernel(const PermParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* ln_m = reinterpret_cast<double*>(smem_raw);                      // [8]
    uint32_t* keys = reinterpret_cast<uint32_t*>(smem_raw + 8 * sizeof(double));   // [N][blockDim.x]
    const int T = blockDim.x, tid = threadIdx.x, N = p.N;
    if (tid < 8) ln_m[tid] = tid == 0 ? -CUDART_INF : log((double)tid);
    __syncthreads();
    const double ln2 = log(2.0);
    uint16_t st_n[kMaxDepth];
    double st_w[kMaxDepth];
    Sums st_s[kMaxDepth];

    // per-lane state of the tour being run; n == 0: the lane needs a new tour
    unsigned long long idx = 0;
    uint32_t c_lo = 0, c_hi = 0, node = 0;
    int n = 0, sp = 0;
    double lnW = 0.0, S = 0.0, SR = 0.0, SG = 0.0;
    bool capped = false;
    uint64_t dg = 0;
    Sums sm = {0, 0, 0, 0};

    // ONE loop for everything: an iteration is one node of every lane's current tour (a growth step, a leaf, or the end of
    // the tour with the draw of the next one). Tours differ in size by orders of magnitude; with a loop per tour inside a
    // loop over tours the lanes of a warp would meet again only after the largest of their 32 tours (measured: 3.2 of 32
    // lanes active), here a lane whose tour ends starts the next one in the same iteration.
    for (;;) {
        if (n == 0) {
            idx = atomicAdd(p.ticket, 1ull);                                 // timing dependent; the record is a function of the tour id only
            if (idx >= p.n_tours) break;
            const uint64_t tour = p.tour_offset + idx;
            c_lo = (uint32_t)tour; c_hi = (uint32_t)(tour >> 32);
            keys[tid] = (uint32_t)kBias | ((uint32_t)kBias << kField) | ((uint32_t)kBias << (2 * kField));
            n = 1; sp = 0; node = 0; capped = false;
            lnW = 0.0; S = 0.0; SR = 0.0; SG = 0.0;
            dg = 0xCBF29CE484222325ull;
            sm = Sums{0, 0, 0, 0};
        }
        bool pop = false, over = false;
        const uint32_t h = keys[(n - 1) * T + tid];                          // r_{n-1}
        if (n == N) {
            // leaf: observables from the running sums (integers until the divide)
            const int hx = (int)(h & kFieldMask) - kBias, hy = (int)((h >> kField) & kFieldMask) - kBias, hz = (int)(h >> (2 * kField)) - kBias;
            const double ree2 = (double)(hx * hx + hy * hy + hz * hz);
            const long long sx = sm.sx, sy = sm.sy, sz = sm.sz;
            const double rg2 = (double)((long long)N * (long long)sm.s2 - (sx * sx + sy * sy + sz * sz)) / ((double)N * (double)N);
            const double w = exp(lnW - p.ln_ref);
            S += w; SR += w * ree2; SG += w * rg2;
            pop = true;
        } else if (node >= p.max_nodes) {
            capped = true;
            over = true;
        } else {
            const uint32_t id = node++;
            // L2: neighbours of r_{n-1} occupied by monomers j <= n-2 of the parity of n (Alg. 1 lines 13-17). The packed
            // difference of two keys is +-1, +-2^10 or +-2^20 exactly for the six neighbour sites: a power-of-two test on
            // its magnitude replaces six compares; the direction bit is formed on the rare hit.
            uint32_t occ = 0;
            for (int j = n - 2; j >= 0; j -= 2) {
                const int32_t w = (int32_t)(keys[j * T + tid] - h);
                const uint32_t a = (uint32_t)abs(w);
                if ((a & (a - 1u)) == 0u && (a & 0x00100401u) != 0u) {
                    const uint32_t axis = a == 1u ? 0u : (a == 1024u ? 1u : 2u);
                    occ |= 1u << (2u * axis + (w < 0 ? 1u : 0u));
                }
            }
            const uint32_t m = 6u - (uint32_t)__popc(occ);
            if (m == 0u) {
                dg = fold(dg, 0u, 0xFFu);
                pop = true;
            } else {
                lnW += ln_m[m];
                uint32_t w4[4];
                philox4x32_10(c_lo, c_hi, (id + 1u) >> 2, 0u, p.key0, p.key1, w4);
                const uint32_t q1 = (id + 1u) & 3u;
                const uint32_t u = q1 == 0u ? w4[0] : q1 == 1u ? w4[1] : q1 == 2u ? w4[2] : w4[3];
                const uint32_t sel = __umulhi(u, m);
                const uint32_t fr = ~occ & 63u;
                const int d = (int)__fns(fr, 0u, (int)sel + 1);             // the sel-th free direction in the order +x,-x,+y,-y,+z,-z
                const uint32_t step = 1u << (kField * (d >> 1));
                const uint32_t k = (d & 1) ? h - step : h + step;
                keys[n * T + tid] = k;
                const int x = (int)(k & kFieldMask) - kBias, y = (int)((k >> kField) & kFieldMask) - kBias, z = (int)(k >> (2 * kField)) - kBias;
                sm.sx += x; sm.sy += y; sm.sz += z; sm.s2 += x * x + y * y + z * z;
                uint32_t event = 0;
                if (n + 1 < N) {
                    if (lnW > __ldg(p.ln_hi + n + 1)) {
                        lnW -= ln2; event = 1u;
                        st_n[sp] = (uint16_t)(n + 1); st_w[sp] = lnW; st_s[sp] = sm; ++sp;      // the second copy
                    } else if (lnW < __ldg(p.ln_lo + n + 1)) {
                        uint32_t c4[4];
                        philox4x32_10(c_lo, c_hi, id >> 2, 2u, p.key0, p.key1, c4);
                        const uint32_t q2 = id & 3u;
                        const uint32_t coin = q2 == 0u ? c4[0] : q2 == 1u ? c4[1] : q2 == 2u ? c4[2] : c4[3];
                        if (coin < 0x80000000u) { event = 3u; pop = true; } else { lnW += ln2; event = 2u; }
                    }
                }
                dg = fold(dg, m | (event << 4), (uint32_t)d);
                if (!pop) ++n;
            }
        }
        if (pop) {
            if (sp == 0) over = true;
            else { --sp; n = st_n[sp]; lnW = st_w[sp]; sm = st_s[sp]; }
        }
        if (over) {
            const bool have = S > 0.0;
            ChainRecord r;
            r.lnW = have ? p.ln_ref + log(S) : -CUDART_INF;
            r.ree2 = have ? SR / S : 0.0; r.rg2 = have ? SG / S : 0.0;
            r.steps = node; r.alive = (have ? 1u : 0u) | (capped ? 2u : 0u); r.digest = dg;
            p.rec[idx] = r;
            n = 0;
        }
    }
}

}  // namespace

int launch_lattice_perm(const PermParams& p, cudaStream_t stream, const char** kernel_name)
{
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    int threads = 128;
    while (threads > 32 && 64 + (size_t)p.N * 4 * threads > (size_t)(64 * 1024)) threads >>= 1;
    const size_t smem = 64 + (size_t)p.N * 4 * threads;
    if (cudaFuncSetAttribute(lattice_perm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -3;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lattice_perm_kernel, threads, smem) != cudaSuccess || per_sm < 1) return -3;
    const uint64_t want = (p.n_tours + threads - 1) / threads, cap = (uint64_t)n_sm * per_sm;
    *kernel_name = "lattice_perm_kernel";
    lattice_perm_kernel<<<(int)(want < cap ? want : cap), threads, smem, stream>>>(p);
    if (cudaGetLastError() != cudaSuccess) return -3;
    const int rr = launch_reduce_records(p.rec, p.n_tours, p.chunk, p.n_vblocks, 0.0, p.lmax, p.out, p.partials, stream);
    return rr < 0 ? rr : 1 + rr;
}

}  // namespace rosen
