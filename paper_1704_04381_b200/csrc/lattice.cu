// lattice.cu -- cubic-lattice Rosenbluth chain generation for sm_100a (steps L0-L5 of DESIGN.md 2;
// PAPER.md:88-179, Algorithm 1; weight Eq. 3 :58). One thread grows one chain at a time; the chain
// lives in shared memory as one packed key per monomer, split by monomer parity, because on a
// bipartite lattice only monomers j with j = s (mod 2) can sit next to the growth point r_{s-1}: the
// scan of Alg. 1 lines 13-17 / 26-31 touches floor(s/2) keys instead of s-1 (exactly the same decisions).
//
// The scan is the hot loop and is hand-scheduled in PTX: per 16-byte shared-memory
// load (4 keys) it runs predicate-chained ISETP.EQ.OR compares -- one instruction per (key, neighbour)
// pair, on the half-rate `alu` pipe -- and, for chains of N <= 128, moves the +-z neighbours to the
// full-rate fp32 lanes: keys are stored as exactly representable floats, and prod_j (key_j - n_d) is zero
// (or NaN after an overflow to inf) iff some key equals the neighbour key n_d. Both tests are exact.
#include <algorithm>
#include <math_constants.h>
#include "common.cuh"
#include "philox.cuh"
#include "reduce.cuh"

namespace rosen {

namespace {

// ---- packed site keys ---------------------------------------------------------------------------
// MIX  (N <= 128): 8-bit fields biased by 128, key < 2^24, stored as the fp32 number of that value.
// !MIX (N <= 512): 10-bit fields biased by 512, stored as the integer itself.
template <bool MIX> struct Key;
template <> struct Key<true>  { static constexpr int kBits = 8,  kBias = 128; };
template <> struct Key<false> { static constexpr int kBits = 10, kBias = 512; };

struct LatTables {
    uint2    lut[64];   // index = occupied-direction mask. .x: bits 0-2 = m, bits 4+4i..6+4i = i-th free direction
                        // (so that (x >> 4*sel) & 0x70 is the byte offset of step[dir]); .y: histogram increment
                        // 1 << 8*(m-2) for m = 2..5, else 0 (m = 1 adds ln 1 = 0, m = 6 happens at s = 1 only)
    int4     step[8];   // per direction: {key delta (float bits if MIX, else int), dx, dy, dz}
    double   ln_m[8];   // ln m; ln_m[0] = -inf (dead)
};

template <bool MIX>
__device__ __forceinline__ void build_tables(LatTables* t)
{
    for (int occ = threadIdx.x; occ < 64; occ += blockDim.x) {
        uint32_t e = 0, m = 0;
        for (int d = 0; d < 6; ++d)
            if (!((occ >> d) & 1)) { e |= (uint32_t)d << (4 + 4 * m); ++m; }
        t->lut[occ] = make_uint2(e | m, (m >= 2 && m <= 5) ? 1u << (8 * (m - 2)) : 0u);
    }
    if (threadIdx.x < 8) {
        const int d = threadIdx.x;
        const int ax = d >> 1, sg = (d & 1) ? -1 : 1;
        int4 s = make_int4(0, 0, 0, 0);
        if (d < 6) {
            const int delta = sg * (1 << (Key<MIX>::kBits * ax));
            s.x = MIX ? __float_as_int((float)delta) : delta;
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
// plus 4 words so that stride/4 is odd (LDS.128 of a quarter-warp is bank-conflict free) and the
// scan's one-chunk-ahead prefetch stays inside the thread's own region.
__host__ __device__ inline int half4_of(int N) { return (((N + 1) / 2) + 3) & ~3; }
__host__ __device__ inline int stride_of(int N) { return 2 * half4_of(N) + 4; }

// ---- L2: the scan ---------------------------------------------------------------------------------
// addr: shared-memory byte address of the parity array; T >= 1 chunks of 4 keys; n0..n5: neighbour
// keys in the order +x,-x,+y,-y,+z,-z. Returns the 6-bit mask of occupied neighbours. Unused slots
// hold 0, which no neighbour key equals. Chunks are double-buffered (a*/b*) so that the next LDS.128
// is in flight while the current 4 keys are tested; the first chunk is peeled so that it initialises
// the predicate chains and the fp32 products instead of separate set-up instructions. The loads run
// at most one chunk past the T-th, which stays inside the thread's own region (stride_of).
#define ROSEN_MIX_KEY(w)                                                                             \
    "setp.eq.or.b32 p0, " #w ", %3, p0; setp.eq.or.b32 p1, " #w ", %4, p1;\n"                         \
    "setp.eq.or.b32 p2, " #w ", %5, p2; setp.eq.or.b32 p3, " #w ", %6, p3;\n"
#define ROSEN_MIX_FP(w, acc4, acc5)                                                                  \
    "sub.rn.f32 t4, " #w ", %7; sub.rn.f32 t5, " #w ", %8;\n"                                         \
    "mul.rn.f32 " #acc4 ", " #acc4 ", t4; mul.rn.f32 " #acc5 ", " #acc5 ", t5;\n"
#define ROSEN_MIX_CHUNK(W)                                                                           \
    ROSEN_MIX_KEY(W##0) ROSEN_MIX_FP(W##0, e4, e5) ROSEN_MIX_KEY(W##1) ROSEN_MIX_FP(W##1, f4, f5)     \
    ROSEN_MIX_KEY(W##2) ROSEN_MIX_FP(W##2, e4, e5) ROSEN_MIX_KEY(W##3) ROSEN_MIX_FP(W##3, f4, f5)
#define ROSEN_MIX_FIRST(W)                                                                           \
    "setp.eq.b32 p0, " #W "0, %3; setp.eq.b32 p1, " #W "0, %4; setp.eq.b32 p2, " #W "0, %5; setp.eq.b32 p3, " #W "0, %6;\n" \
    "sub.rn.f32 e4, " #W "0, %7; sub.rn.f32 e5, " #W "0, %8; sub.rn.f32 f4, " #W "1, %7; sub.rn.f32 f5, " #W "1, %8;\n"     \
    ROSEN_MIX_KEY(W##1) ROSEN_MIX_KEY(W##2) ROSEN_MIX_FP(W##2, e4, e5) ROSEN_MIX_KEY(W##3) ROSEN_MIX_FP(W##3, f4, f5)

__device__ __forceinline__ uint32_t scan_mix(uint32_t addr, uint32_t T, uint32_t n0, uint32_t n1, uint32_t n2,
                                             uint32_t n3, uint32_t n4, uint32_t n5)
{
    uint32_t occ;
    asm volatile("{\n"
        ".reg .pred p0, p1, p2, p3, q;\n"
        ".reg .b32 a0, a1, a2, a3, b0, b1, b2, b3, ad, cnt, r0, r1, r2, r3, r4, r5;\n"
        ".reg .f32 e4, e5, f4, f5, t4, t5;\n"
        "mov.u32 ad, %1; mov.u32 cnt, %2;\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad];\n"
        "ld.shared.v4.b32 {b0, b1, b2, b3}, [ad+16];\n"
        ROSEN_MIX_FIRST(a)
        "setp.eq.u32 q, cnt, 1;\n"
        "@q bra SCAN_DONE;\n"
        "SCAN_LOOP:\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad+32];\n"
        ROSEN_MIX_CHUNK(b)
        "setp.eq.u32 q, cnt, 2;\n"
        "@q bra SCAN_DONE;\n"
        "ld.shared.v4.b32 {b0, b1, b2, b3}, [ad+48];\n"
        ROSEN_MIX_CHUNK(a)
        "add.u32 ad, ad, 32; sub.u32 cnt, cnt, 2;\n"
        "setp.ne.u32 q, cnt, 1;\n"
        "@q bra SCAN_LOOP;\n"
        "SCAN_DONE:\n"
        "mul.rn.f32 e4, e4, f4; mul.rn.f32 e5, e5, f5;\n"
        "selp.u32 r0, 1, 0, p0; selp.u32 r1, 2, 0, p1; selp.u32 r2, 4, 0, p2; selp.u32 r3, 8, 0, p3;\n"
        "setp.equ.f32 p0, e4, 0f00000000; setp.equ.f32 p1, e5, 0f00000000;\n"   // zero, or NaN = inf * 0
        "selp.u32 r4, 16, 0, p0; selp.u32 r5, 32, 0, p1;\n"
        "add.u32 r0, r0, r1; add.u32 r2, r2, r3; add.u32 r4, r4, r5;\n"
        "add.u32 r0, r0, r2; add.u32 %0, r0, r4;\n"
        "}\n"
        : "=r"(occ)
        : "r"(addr), "r"(T), "r"(n0), "r"(n1), "r"(n2), "r"(n3), "r"(n4), "r"(n5)
        : "memory");
    return occ;
}

#define ROSEN_INT_KEY(w)                                                                             \
    "setp.eq.or.b32 p0, " #w ", %3, p0; setp.eq.or.b32 p1, " #w ", %4, p1; setp.eq.or.b32 p2, " #w ", %5, p2;\n" \
    "setp.eq.or.b32 p3, " #w ", %6, p3; setp.eq.or.b32 p4, " #w ", %7, p4; setp.eq.or.b32 p5, " #w ", %8, p5;\n"
#define ROSEN_INT_CHUNK(W) ROSEN_INT_KEY(W##0) ROSEN_INT_KEY(W##1) ROSEN_INT_KEY(W##2) ROSEN_INT_KEY(W##3)
#define ROSEN_INT_FIRST(W)                                                                           \
    "setp.eq.b32 p0, " #W "0, %3; setp.eq.b32 p1, " #W "0, %4; setp.eq.b32 p2, " #W "0, %5;\n"        \
    "setp.eq.b32 p3, " #W "0, %6; setp.eq.b32 p4, " #W "0, %7; setp.eq.b32 p5, " #W "0, %8;\n"        \
    ROSEN_INT_KEY(W##1) ROSEN_INT_KEY(W##2) ROSEN_INT_KEY(W##3)

__device__ __forceinline__ uint32_t scan_int(uint32_t addr, uint32_t T, uint32_t n0, uint32_t n1, uint32_t n2,
                                             uint32_t n3, uint32_t n4, uint32_t n5)
{
    uint32_t occ;
    asm volatile("{\n"
        ".reg .pred p0, p1, p2, p3, p4, p5, q;\n"
        ".reg .b32 a0, a1, a2, a3, b0, b1, b2, b3, ad, cnt, r0, r1, r2, r3, r4, r5;\n"
        "mov.u32 ad, %1; mov.u32 cnt, %2;\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad];\n"
        "ld.shared.v4.b32 {b0, b1, b2, b3}, [ad+16];\n"
        ROSEN_INT_FIRST(a)
        "setp.eq.u32 q, cnt, 1;\n"
        "@q bra SCAN_DONE;\n"
        "SCAN_LOOP:\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad+32];\n"
        ROSEN_INT_CHUNK(b)
        "setp.eq.u32 q, cnt, 2;\n"
        "@q bra SCAN_DONE;\n"
        "ld.shared.v4.b32 {b0, b1, b2, b3}, [ad+48];\n"
        ROSEN_INT_CHUNK(a)
        "add.u32 ad, ad, 32; sub.u32 cnt, cnt, 2;\n"
        "setp.ne.u32 q, cnt, 1;\n"
        "@q bra SCAN_LOOP;\n"
        "SCAN_DONE:\n"
        "selp.u32 r0, 1, 0, p0; selp.u32 r1, 2, 0, p1; selp.u32 r2, 4, 0, p2;\n"
        "selp.u32 r3, 8, 0, p3; selp.u32 r4, 16, 0, p4; selp.u32 r5, 32, 0, p5;\n"
        "add.u32 r0, r0, r1; add.u32 r2, r2, r3; add.u32 r4, r4, r5;\n"
        "add.u32 r0, r0, r2; add.u32 %0, r0, r4;\n"
        "}\n"
        : "=r"(occ)
        : "r"(addr), "r"(T), "r"(n0), "r"(n1), "r"(n2), "r"(n3), "r"(n4), "r"(n5)
        : "memory");
    return occ;
}

template <bool MIX>
__device__ __forceinline__ uint32_t key_add(uint32_t h, int delta_key)
{
    return MIX ? __float_as_uint(__fadd_rn(__uint_as_float(h), __int_as_float(delta_key))) : h + (uint32_t)delta_key;
}

// key delta of +1 along axis ax, in the key's own encoding
template <bool MIX>
__device__ __forceinline__ constexpr int unit_delta(int ax)
{
    return 1 << (Key<MIX>::kBits * ax);
}

template <bool MIX, bool DIGEST, bool TRAJ>
__global__ void __launch_bounds__(256) lattice_kernel(const LatticeParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    LatTables* tab = reinterpret_cast<LatTables*>(smem_raw);
    Partial* scratch = reinterpret_cast<Partial*>(smem_raw + sizeof(LatTables));
    uint32_t* chains = reinterpret_cast<uint32_t*>(smem_raw + sizeof(LatTables) + 8 * sizeof(Partial));

    constexpr int kBits = Key<MIX>::kBits, kBias = Key<MIX>::kBias;
    constexpr uint32_t kFieldMask = (1u << kBits) - 1u;
    constexpr uint32_t kOriginInt = (uint32_t)kBias | ((uint32_t)kBias << kBits) | ((uint32_t)kBias << (2 * kBits));
    const uint32_t kOrigin = MIX ? __float_as_uint((float)kOriginInt) : kOriginInt;
    // neighbour key offsets (compile-time constants in the key's encoding)
    const uint32_t dxp = MIX ? __float_as_uint(1.0f) : 1u;
    (void)dxp;

    const int N = p.N;
    const int half4 = half4_of(N), stride = stride_of(N);
    uint32_t* ev = chains + (size_t)threadIdx.x * stride;   // monomers 0,2,4,...
    uint32_t* od = ev + half4;                              // monomers 1,3,5,...
    const uint32_t ev_addr = (uint32_t)__cvta_generic_to_shared(ev);
    const uint32_t od_addr = ev_addr + (uint32_t)half4 * 4u;

    build_tables<MIX>(tab);
    __syncthreads();

    const uint32_t per_thread = p.chunk / blockDim.x;       // chunk is a multiple of 256 >= blockDim.x

    for (uint32_t vb = blockIdx.x; vb < p.n_vblocks; vb += gridDim.x) {
        Partial acc = partial_zero();
        for (uint32_t it = 0; it < per_thread; ++it) {
            const uint64_t idx = (uint64_t)vb * p.chunk + (uint64_t)it * blockDim.x + threadIdx.x;
            if (idx >= p.n_chains) break;
            const uint64_t chain = p.chain_offset + idx;
            const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);

            // L0: r_0 = origin, lnW = 0, alive. Unused words hold 0, which no neighbour key can equal.
            for (int i = 0; i < stride / 4; ++i) reinterpret_cast<uint4*>(ev)[i] = make_uint4(0, 0, 0, 0);
            ev[0] = kOrigin;
            uint32_t h = kOrigin;
            int hx = 0, hy = 0, hz = 0, sx = 0, sy = 0, sz = 0, s2 = 0;
            double lnW = 0.0;
            uint32_t hist = 0;                 // MIX: counts of m = 2,3,4,5 in bytes 0..3
            uint32_t alive_i = 1u;
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
                    uint32_t occ = 0;
                    const uint32_t T = (uint32_t)(((s >> 1) + 3) >> 2);
                    if (T != 0u) {
                        const uint32_t n0 = key_add<MIX>(h, MIX ? __float_as_int(1.0f) : 1);
                        const uint32_t n1 = key_add<MIX>(h, MIX ? __float_as_int(-1.0f) : -1);
                        const uint32_t n2 = key_add<MIX>(h, MIX ? __float_as_int((float)(1 << kBits)) : (1 << kBits));
                        const uint32_t n3 = key_add<MIX>(h, MIX ? __float_as_int(-(float)(1 << kBits)) : -(1 << kBits));
                        const uint32_t n4 = key_add<MIX>(h, MIX ? __float_as_int((float)(1 << (2 * kBits))) : (1 << (2 * kBits)));
                        const uint32_t n5 = key_add<MIX>(h, MIX ? __float_as_int(-(float)(1 << (2 * kBits))) : -(1 << (2 * kBits)));
                        const uint32_t addr = (k & 1) ? od_addr : ev_addr;
                        occ = MIX ? scan_mix(addr, T, n0, n1, n2, n3, n4, n5) : scan_int(addr, T, n0, n1, n2, n3, n4, n5);
                    }
                    const uint2 le = tab->lut[occ];
                    const uint32_t e = le.x;
                    const uint32_t m = e & 7u;

                    // L3: weight. MIX: histogram of m (packed 8-bit counts, N <= 128), lnW assembled once per
                    // chain; else lnW += ln m with ln_m[0] = -inf. alive_i = 1 until the first m = 0.
                    steps += alive_i;
                    if (MIX) hist += le.y; else lnW += tab->ln_m[m];
                    if (TRAJ && mrow) mrow[s - 1] = alive_i ? (uint8_t)m : (uint8_t)0;

                    // L4: uniform choice among the free neighbours, then place monomer s
                    const uint32_t sel = __umulhi(w[k], m);
                    const uint32_t off = (e >> (4u * sel)) & 0x70u;          // 16 * direction
                    if (DIGEST) { if (alive_i) dg = digest_fold(dg, m, m ? (off >> 4) : 0xFFu); }
                    alive_i &= min(m, 1u);
                    const int4 st = *reinterpret_cast<const int4*>(reinterpret_cast<const unsigned char*>(tab->step) + off);
                    h = key_add<MIX>(h, st.x); hx += st.y; hy += st.z; hz += st.w;
                    ((k & 1) ? od : ev)[s >> 1] = h;

                    // L5: running sums for Rg^2
                    sx += hx; sy += hy; sz += hz; s2 += hx * hx + hy * hy + hz * hz;
                }
            }

            // L5: per-chain observables (integers until the final divide)
            const bool alive = alive_i != 0u;
            if (MIX) {   // lnW = ln 6 + sum_m count_m ln m, fixed order (the first step always has m = 6)
                lnW = tab->ln_m[6];
                lnW += (double)(hist & 255u) * tab->ln_m[2];
                lnW += (double)((hist >> 8) & 255u) * tab->ln_m[3];
                lnW += (double)((hist >> 16) & 255u) * tab->ln_m[4];
                lnW += (double)(hist >> 24) * tab->ln_m[5];
                if (!alive) lnW = -CUDART_INF;
            }
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
                // D1 (lattice): each thread unpacks and writes its own chain; monomers from the death
                // step on are zero. steps = death step for a dead chain.
                int32_t* c = reinterpret_cast<int32_t*>(p.out.conf) + idx * (uint64_t)N * 3;
                const int placed = alive ? N : (int)steps;
                for (int i = 0; i < N; ++i) {
                    const uint32_t raw = ((i & 1) ? od : ev)[i >> 1];
                    const uint32_t v = MIX ? (uint32_t)__float2int_rn(__uint_as_float(raw)) : raw;
                    const bool ok = i < placed;
                    c[3 * i + 0] = ok ? (int)(v & kFieldMask) - kBias : 0;
                    c[3 * i + 1] = ok ? (int)((v >> kBits) & kFieldMask) - kBias : 0;
                    c[3 * i + 2] = ok ? (int)((v >> (2 * kBits)) & kFieldMask) - kBias : 0;
                }
            }
        }
        block_reduce_store(acc, scratch, p.partials + vb);
    }
}

// =====================================================================================================
// N <= 64: the byte-dot-product scan. Keys are plain integers with three 8-bit fields
// biased by 128, so w = key_j - h is the integer dx + 256 dy + 65536 dz with |d| <= 126 < 2^7, a unique
// balanced representation: monomer j sits on a neighbour site of h iff |w| is 1, 2^8 or 2^16, i.e. iff
// exactly one byte of |w| is 1 and the rest are 0 (|w| < 2^24), i.e. iff dp4a.u8(|w|, |w|) == 1. The
// scan XOR-accumulates w over those keys without a predicate: d = dp4a(|w|,|w|,-1) is 0 for a
// neighbour and >= 1 otherwise, and w >> (32 d) keeps w or clears it (PTX shr clamps at 32). Every
// neighbour site holds at most one monomer, so the XOR of {1, -1, 256, -256, 65536, -65536} over the
// occupied subset decodes uniquely from bits 0,1,8,9,16,17 (table index, build_dp_tables).
// Per key: IADD, IABS, IDP.4A, IMAD.SHL, SHF, 1/2 LOP3 -- 5.5 issue slots against 8 for the compare scan.
// -----------------------------------------------------------------------------------------------------
struct DpTables {
    uint2    lut[64];   // index = (b0,b1,b8,b9,b16,b17) of the XOR. .x: bits 0-2 = m, bits 4+4i..6+4i = i-th free
                        // direction; .y: histogram increment 1 << 8*(m-2) for m = 2..5
    int32_t  delta[8];  // key delta per direction
    double   ln_m[8];
};

__device__ __forceinline__ void build_dp_tables(DpTables* t)
{
    for (int idx = threadIdx.x; idx < 64; idx += blockDim.x) {
        const int b0 = idx & 1, b1 = (idx >> 1) & 1, b8 = (idx >> 2) & 1, b9 = (idx >> 3) & 1, b16 = (idx >> 4) & 1, b17 = (idx >> 5) & 1;
        // XOR patterns: +x 0x1, -x 0xFFFFFFFF, +y 0x100, -y 0xFFFFFF00, +z 0x10000, -z 0xFFFF0000
        const int occ_d[6] = { b0 ^ b1, b1, b8 ^ b9, b9 ^ b1, b16 ^ b17, b17 ^ b9 };
        uint32_t e = 0, m = 0;
        for (int d = 0; d < 6; ++d)
            if (!occ_d[d]) { e |= (uint32_t)d << (4 + 4 * m); ++m; }
        t->lut[idx] = make_uint2(e | m, (m >= 2 && m <= 5) ? 1u << (8 * (m - 2)) : 0u);
    }
    if (threadIdx.x < 8) {
        const int d = threadIdx.x;
        t->delta[d] = d < 6 ? ((d & 1) ? -1 : 1) * (1 << (8 * (d >> 1))) : 0;
        t->ln_m[d] = d == 0 ? -CUDART_INF : log((double)d);
    }
}

#define ROSEN_DP_CHUNK(W)                                                                            \
    "sub.s32 w0, " #W "0, %3; sub.s32 w1, " #W "1, %3; sub.s32 w2, " #W "2, %3; sub.s32 w3, " #W "3, %3;\n" \
    "abs.s32 t0, w0; abs.s32 t1, w1; abs.s32 t2, w2; abs.s32 t3, w3;\n"                                \
    "dp4a.u32.u32 t0, t0, t0, m1; dp4a.u32.u32 t1, t1, t1, m1; dp4a.u32.u32 t2, t2, t2, m1; dp4a.u32.u32 t3, t3, t3, m1;\n" \
    "mul.lo.u32 t0, t0, 32; mul.lo.u32 t1, t1, 32; mul.lo.u32 t2, t2, 32; mul.lo.u32 t3, t3, 32;\n"    \
    "shr.u32 w0, w0, t0; shr.u32 w1, w1, t1; shr.u32 w2, w2, t2; shr.u32 w3, w3, t3;\n"                \
    "lop3.b32 A, A, w0, w1, 0x96; lop3.b32 A, A, w2, w3, 0x96;\n"

// addr: shared byte address of the parity array, T >= 1 chunks of 4 keys, h: key of r_{s-1}. Returns the XOR.
// Chunks are double-buffered; the load runs at most one chunk past the T-th (inside the thread's own region).
__device__ __forceinline__ uint32_t scan_dp(uint32_t addr, uint32_t T, uint32_t h)
{
    uint32_t A;
    asm volatile("{\n"
        ".reg .pred q;\n"
        ".reg .b32 a0, a1, a2, a3, b0, b1, b2, b3, ad, cnt, A, m1, w0, w1, w2, w3, t0, t1, t2, t3;\n"
        "mov.u32 ad, %1; mov.u32 cnt, %2; mov.u32 A, 0; mov.u32 m1, 0xFFFFFFFF;\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad];\n"
        "DP_LOOP:\n"
        "ld.shared.v4.b32 {b0, b1, b2, b3}, [ad+16];\n"
        ROSEN_DP_CHUNK(a)
        "setp.eq.u32 q, cnt, 1;\n"
        "@q bra DP_DONE;\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad+32];\n"
        ROSEN_DP_CHUNK(b)
        "add.u32 ad, ad, 32; sub.u32 cnt, cnt, 2;\n"
        "setp.ne.u32 q, cnt, 0;\n"
        "@q bra DP_LOOP;\n"
        "DP_DONE:\n"
        "mov.u32 %0, A;\n"
        "}\n"
        : "=r"(A)
        : "r"(addr), "r"(T), "r"(h)
        : "memory");
    return A;
}

__device__ __forceinline__ uint2 lds64(uint32_t a) { uint2 v; asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds32(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts128(uint32_t a, uint32_t v) { asm volatile("st.shared.v4.u32 [%0], {%1, %2, %2, %2};" :: "r"(a), "r"(v), "r"(0u) : "memory"); }

template <bool DIGEST, bool TRAJ>
__global__ void __launch_bounds__(256) lattice_dp_kernel(const LatticeParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    DpTables* tab = reinterpret_cast<DpTables*>(smem_raw);
    Partial* scratch = reinterpret_cast<Partial*>(smem_raw + sizeof(DpTables));
    uint32_t* chains = reinterpret_cast<uint32_t*>(smem_raw + sizeof(DpTables) + 8 * sizeof(Partial));

    constexpr uint32_t kOrigin = 0x00808080u;
    const int N = p.N;
    const int half4 = half4_of(N), stride = stride_of(N);
    uint32_t* ev = chains + (size_t)threadIdx.x * stride;   // monomers 0,2,4,...
    uint32_t* od = ev + half4;                              // monomers 1,3,5,...
    const uint32_t lut_addr = (uint32_t)__cvta_generic_to_shared(tab->lut);
    const uint32_t delta_addr = (uint32_t)__cvta_generic_to_shared(tab->delta);
    const uint32_t ev_addr = (uint32_t)__cvta_generic_to_shared(ev);
    const uint32_t od_addr = ev_addr + (uint32_t)half4 * 4u;

    build_dp_tables(tab);
    __syncthreads();

    const uint32_t per_thread = p.chunk / blockDim.x;

    for (uint32_t vb = blockIdx.x; vb < p.n_vblocks; vb += gridDim.x) {
        Partial acc = partial_zero();
        for (uint32_t it = 0; it < per_thread; ++it) {
            const uint64_t idx = (uint64_t)vb * p.chunk + (uint64_t)it * blockDim.x + threadIdx.x;
            if (idx >= p.n_chains) break;
            const uint64_t chain = p.chain_offset + idx;
            const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);

            // L0. No clearing pass: the first key of every 4-key chunk is stored as {key, 0, 0, 0}, so a scan
            // never sees a key of the previous chain (0 is not a neighbour of any head: |0 - h| >= 0x414141).
            uint32_t h = kOrigin;
            sts128(ev_addr, h);
            int sx = 0, sy = 0, sz = 0, s2 = 0;
            uint32_t hist = 0, alive_i = 1u, steps = 0;
            uint64_t dg = 0xCBF29CE484222325ull;
            uint8_t* mrow = TRAJ && p.out.m_seq ? p.out.m_seq + idx * (uint64_t)(N - 1) : nullptr;

            for (int q = 0; 4 * q < N; ++q) {
                uint32_t w[4];
                philox4x32_10(c_lo, c_hi, (uint32_t)q, 0u, p.key0, p.key1, w);   // L1
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int s = 4 * q + k;
                    if (s == 0 || s >= N) continue;

                    // L2
                    uint32_t A = 0;
                    const uint32_t T = (uint32_t)(((s >> 1) + 3) >> 2);
                    if (T != 0u) A = scan_dp((k & 1) ? od_addr : ev_addr, T, h);
                    const uint32_t li = (((A & 0x00030303u) * 0x00010410u) >> 13) & 0x1F8u;   // 8 * (b0,b1,b8,b9,b16,b17)
                    const uint2 le = lds64(lut_addr + li);
                    const uint32_t m = le.x & 7u;

                    // L3
                    steps += alive_i;
                    hist += le.y;
                    if (TRAJ && mrow) mrow[s - 1] = alive_i ? (uint8_t)m : (uint8_t)0;

                    // L4
                    const uint32_t sel = __umulhi(w[k], m);
                    const uint32_t d4 = (le.x >> (4u * sel + 2u)) & 0x1Cu;     // 4 * direction
                    if (DIGEST) { if (alive_i) dg = digest_fold(dg, m, m ? (d4 >> 2) : 0xFFu); }
                    alive_i &= min(m, 1u);
                    h += lds32(delta_addr + d4);
                    const uint32_t slot = ((k & 1) ? od_addr : ev_addr) + 4u * (uint32_t)(s >> 1);
                    if (((s >> 1) & 3) == 0) sts128(slot, h); else sts32(slot, h);

                    // L5: signed bytes of r_s; |r|^2 and the three coordinate sums as byte dot products
                    const int sg = (int)(h ^ kOrigin);
                    s2 = __dp4a(sg, sg, s2);
                    sx = __dp4a(sg, 0x00000001, sx); sy = __dp4a(sg, 0x00000100, sy); sz = __dp4a(sg, 0x00010000, sz);
                }
            }

            const bool alive = alive_i != 0u;
            double lnW = tab->ln_m[6];
            lnW += (double)(hist & 255u) * tab->ln_m[2];
            lnW += (double)((hist >> 8) & 255u) * tab->ln_m[3];
            lnW += (double)((hist >> 16) & 255u) * tab->ln_m[4];
            lnW += (double)(hist >> 24) * tab->ln_m[5];
            if (!alive) lnW = -CUDART_INF;
            double ree2 = 0.0, rg2 = 0.0;
            if (alive) {
                const int sg = (int)(h ^ kOrigin);
                ree2 = (double)__dp4a(sg, sg, 0);
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
                int32_t* c = reinterpret_cast<int32_t*>(p.out.conf) + idx * (uint64_t)N * 3;
                const int placed = alive ? N : (int)steps;
                for (int i = 0; i < N; ++i) {
                    const uint32_t v = ((i & 1) ? od : ev)[i >> 1];
                    const bool ok = i < placed;
                    c[3 * i + 0] = ok ? (int)(v & 255u) - 128 : 0;
                    c[3 * i + 1] = ok ? (int)((v >> 8) & 255u) - 128 : 0;
                    c[3 * i + 2] = ok ? (int)((v >> 16) & 255u) - 128 : 0;
                }
            }
        }
        block_reduce_store(acc, scratch, p.partials + vb);
    }
}

template <typename Kern>
int launch_kernel(Kern kern, size_t table_bytes, const LatticeParams& p, cudaStream_t stream, int* grid_out)
{
    int dev = 0, n_sm = 0, smem_max = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t fixed = table_bytes + 8 * sizeof(Partial);
    const size_t per_thread = (size_t)stride_of(p.N) * 4;
    // threads per block depends on N only (never on the output variant): it fixes the reduction tree.
    int threads = 256;
    while (threads > 32 && fixed + per_thread * threads > (size_t)(72 * 1024)) threads >>= 1;
    const size_t smem = fixed + per_thread * threads;
    if (smem > (size_t)smem_max) return -2;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -3;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) return -3;
    // One resident wave; virtual blocks (common.cuh) are strided over it, so the grid is free to follow
    // the real occupancy of this variant without touching the sums.
    const uint32_t cap = (uint32_t)n_sm * (uint32_t)per_sm;
    const int grid = (int)(p.n_vblocks < cap ? p.n_vblocks : cap);
    kern<<<grid, threads, smem, stream>>>(p);
    if (cudaGetLastError() != cudaSuccess) return -3;
    *grid_out = grid;
    return 1;
}

template <bool MIX, bool DIGEST, bool TRAJ>
int launch_variant(const LatticeParams& p, cudaStream_t stream, int* grid_out)
{
    return launch_kernel(lattice_kernel<MIX, DIGEST, TRAJ>, sizeof(LatTables), p, stream, grid_out);
}

int launch_dp(const LatticeParams& p, cudaStream_t stream, int* grid_out)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    const size_t tb = sizeof(DpTables);
    if (traj) return digest ? launch_kernel(lattice_dp_kernel<true, true>, tb, p, stream, grid_out)
                            : launch_kernel(lattice_dp_kernel<false, true>, tb, p, stream, grid_out);
    return digest ? launch_kernel(lattice_dp_kernel<true, false>, tb, p, stream, grid_out)
                  : launch_kernel(lattice_dp_kernel<false, false>, tb, p, stream, grid_out);
}

template <bool MIX>
int launch_mix(const LatticeParams& p, cudaStream_t stream, int* grid_out)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    if (traj) return digest ? launch_variant<MIX, true, true>(p, stream, grid_out) : launch_variant<MIX, false, true>(p, stream, grid_out);
    return digest ? launch_variant<MIX, true, false>(p, stream, grid_out) : launch_variant<MIX, false, false>(p, stream, grid_out);
}

}  // namespace

int launch_lattice(const LatticeParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    if (p.N <= 64) {    // |dx|,|dy|,|dz| <= 126 fit signed bytes: byte-dot-product scan
        *kernel_name = traj ? (digest ? "lattice_dp_kernel<digest,traj>" : "lattice_dp_kernel<traj>")
                            : (digest ? "lattice_dp_kernel<digest>" : "lattice_dp_kernel");
        return launch_dp(p, stream, grid_out);
    }
    if (p.N <= 128) {   // keys < 2^24 are exact in fp32: mixed ISETP / fp32-product scan
        *kernel_name = traj ? (digest ? "lattice_kernel<mix,digest,traj>" : "lattice_kernel<mix,traj>")
                            : (digest ? "lattice_kernel<mix,digest>" : "lattice_kernel<mix>");
        return launch_mix<true>(p, stream, grid_out);
    }
    *kernel_name = traj ? (digest ? "lattice_kernel<int,digest,traj>" : "lattice_kernel<int,traj>")
                        : (digest ? "lattice_kernel<int,digest>" : "lattice_kernel<int>");
    return launch_mix<false>(p, stream, grid_out);
}

}  // namespace rosen
