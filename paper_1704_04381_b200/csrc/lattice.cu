// lattice.cu -- cubic-lattice Rosenbluth chain generation for sm_100a (steps L0-L5 of DESIGN.md 2;
// PAPER.md:88-179, Algorithm 1; weight Eq. 3 :58). One thread grows one chain at a time; the chain
// lives in shared memory as one packed key per monomer, split by monomer parity, because on a
// bipartite lattice only monomers j with j = s (mod 2) can sit next to the growth point r_{s-1}: the
// scan of Alg. 1 lines 13-17 / 26-31 touches floor(s/2) keys instead of s-1 (exactly the same decisions).
//
// The scan is the hot loop and is hand-scheduled in PTX. It never compares a key with the six
// neighbour keys: it classifies w = key_j - h (an integer, because the fields cannot borrow into each other for
// chains this short) with a byte dot product on the tensor-free IDP.4A path and XOR-accumulates the neighbours'
// w (half of the keys select by a clamped shift, half by a predicate: that balances the alu and fma-heavy pipes)
// -- about 5.25 issue slots per key (N <= 128) or 7.25 (N <= 512) instead of 6 half-rate ISETP.
#include <algorithm>
#include <math_constants.h>
#include "common.cuh"
#include "philox.cuh"
#include "reduce.cuh"

namespace rosen {

namespace {

__device__ __forceinline__ uint64_t digest_fold(uint64_t h, uint32_t m, uint32_t choice)
{
    return (h ^ (uint64_t)(m | (choice << 8))) * 0x100000001B3ull;
}

// stride (in 32-bit words) of one thread's chain storage: two parity arrays of half4 words each,
// plus 4 words so that stride/4 is odd (LDS.128 of a quarter-warp is bank-conflict free) and the
// scan's one-chunk-ahead prefetch stays inside the thread's own region.
__host__ __device__ inline int half4_of(int N) { return (((N + 1) / 2) + 3) & ~3; }
__host__ __device__ inline int stride_of(int N) { return 2 * half4_of(N) + 4; }

// =====================================================================================================
// N <= 128: the byte-dot-product scan. Keys are plain integers with three 8-bit fields
// biased by 128 (|coordinate| <= 127), and the scan at step s only meets monomers j <= s-2 <= 125 bonds away from
// the growth point, so w = key_j - h is the integer dx + 256 dy + 65536 dz with |d| <= 126 < 2^7, a unique
// balanced representation: monomer j sits on a neighbour site of h iff |w| is 1, 2^8 or 2^16, i.e. iff
// exactly one byte of |w| is 1 and the rest are 0 (|w| < 2^24), i.e. iff dp4a.u8(|w|, |w|) == 1. The
// scan XOR-accumulates w over those keys without a predicate: d = dp4a(|w|,|w|,-1) is 0 for a
// neighbour and >= 1 otherwise, and w >> (32 d) keeps w or clears it (PTX shr clamps at 32). Every
// neighbour site holds at most one monomer, so the XOR of {1, -1, 256, -256, 65536, -65536} over the
// occupied subset decodes uniquely from bits 0,1,8,9,16,17 (table index, build_dp_tables).
// Per key: IADD, IABS, IDP.4A, then either IMAD.SHL, SHF, 1/2 LOP3 (keys 0, 2 of a chunk) or ISETP, predicated LOP3
// (keys 1, 3) -- 5.25 issue slots against 8 for the compare scan.
// -----------------------------------------------------------------------------------------------------
struct DpTables {
    uint4    lut[64];   // index = (b0,b1,b8,b9,b16,b17) of the XOR. Bytes 0..5 of (.x, .y) = 4 * (i-th free direction), picked
                        // with one byte permute; .z: histogram increment 1 << 8*(m-2) for m = 2..5; .w = m
    int32_t  delta[8];  // key delta per direction; [6], [7]: unused directions, hold the byte selectors 0x100, 0x10000
    double   ln_m[8];
};

template <int B>
__device__ __forceinline__ void build_dp_tables(DpTables* t)
{
    for (int idx = threadIdx.x; idx < 64; idx += blockDim.x) {
        const int b0 = idx & 1, b1 = (idx >> 1) & 1, b8 = (idx >> 2) & 1, b9 = (idx >> 3) & 1, b16 = (idx >> 4) & 1, b17 = (idx >> 5) & 1;
        // XOR patterns: +x 0x1, -x 0xFFFFFFFF, +y 0x100, -y 0xFFFFFF00, +z 0x10000, -z 0xFFFF0000
        const int occ_d[6] = { b0 ^ b1, b1, b8 ^ b9, b9 ^ b1, b16 ^ b17, b17 ^ b9 };
        uint64_t e = 0;
        uint32_t m = 0;
        for (int d = 0; d < 6; ++d)
            if (!occ_d[d]) { e |= (uint64_t)(4 * d) << (8 * m); ++m; }
        t->lut[idx] = make_uint4((uint32_t)e, (uint32_t)(e >> 32), (m >= 2 && m <= 5) ? 1u << (8 * (m - 2)) : 0u, m);
    }
    if (threadIdx.x < 8) {
        const int d = threadIdx.x;
        t->delta[d] = d < 6 ? ((d & 1) ? -1 : 1) * (1 << (B * (d >> 1))) : (d == 6 ? 0x100 : 0x10000);
        t->ln_m[d] = d == 0 ? -CUDART_INF : log((double)d);
    }
}

#define ROSEN_DP_CHUNK(W)                                                                            \
    "sub.s32 w0, " #W "0, %3; sub.s32 w1, " #W "1, %3; sub.s32 w2, " #W "2, %3; sub.s32 w3, " #W "3, %3;\n" \
    "abs.s32 t0, w0; abs.s32 t1, w1; abs.s32 t2, w2; abs.s32 t3, w3;\n"                                \
    "dp4a.u32.u32 t0, t0, t0, m1; dp4a.u32.u32 t1, t1, t1, m1; dp4a.u32.u32 t2, t2, t2, m1; dp4a.u32.u32 t3, t3, t3, m1;\n" \
    "mul.lo.u32 t0, t0, 32; mul.lo.u32 t2, t2, 32;\n"                                                  \
    "shr.u32 w0, w0, t0; shr.u32 w2, w2, t2;\n"                                                        \
    "setp.eq.u32 p1, t1, 0; setp.eq.u32 p3, t3, 0;\n"                                                  \
    "lop3.b32 A, A, w0, w2, 0x96; @p1 xor.b32 A, A, w1; @p3 xor.b32 A, A, w3;\n"

// addr: shared byte address of the parity array, T >= 1 chunks of 4 keys, h: key of r_{s-1}. Returns the XOR.
// Chunks are double-buffered; the load runs at most one chunk past the T-th (inside the thread's own region).
// minus1 = 0xFFFFFFFF in a register that the caller loaded from memory (as an immediate it is re-materialised in every call)
__device__ __forceinline__ uint32_t scan_dp(uint32_t addr, uint32_t T, uint32_t h, uint32_t minus1)
{
    uint32_t A;
    asm volatile("{\n"
        ".reg .pred q, p1, p3;\n"
        ".reg .b32 a0, a1, a2, a3, b0, b1, b2, b3, ad, od, cnt, A, m1, w0, w1, w2, w3, t0, t1, t2, t3;\n"
        "mov.u32 ad, %1; mov.u32 cnt, %2; mov.u32 A, 0; mov.u32 m1, %4;\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad];\n"
        "and.b32 od, cnt, 1;\n"
        "setp.eq.u32 q, od, 0;\n"
        "@q bra DP_EVEN;\n"                      // odd T: peel one chunk, then whole pairs without a mid-loop exit
        ROSEN_DP_CHUNK(a)
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad+16];\n"
        "add.u32 ad, ad, 16; sub.u32 cnt, cnt, 1;\n"
        "DP_EVEN:\n"
        "setp.eq.u32 q, cnt, 0;\n"
        "@q bra DP_DONE;\n"
        "DP_LOOP:\n"
        "ld.shared.v4.b32 {b0, b1, b2, b3}, [ad+16];\n"
        ROSEN_DP_CHUNK(a)
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad+32];\n"
        ROSEN_DP_CHUNK(b)
        "add.u32 ad, ad, 32; sub.u32 cnt, cnt, 2;\n"
        "setp.ne.u32 q, cnt, 0;\n"
        "@q bra DP_LOOP;\n"
        "DP_DONE:\n"
        "mov.u32 %0, A;\n"
        "}\n"
        : "=r"(A)
        : "r"(addr), "r"(T), "r"(h), "r"(minus1)
        : "memory");
    return A;
}

// 128 < N <= 512: 10-bit fields. |w| is 1, 2^10 or 2^20 iff z = |w| & ((|w| - 1) | ~M) is 0 (power of two inside
// M = 2^0 | 2^10 | 2^20; |w| = 0 cannot occur: sites are distinct and an empty slot gives |w| = h). d = byte sum of z
// (IDP.4A against 0x01010101) is 0 for a neighbour and >= 1 otherwise; the rest is as in scan_dp.
#define ROSEN_DPW_CHUNK(W)                                                                           \
    "sub.s32 w0, " #W "0, %3; sub.s32 w1, " #W "1, %3; sub.s32 w2, " #W "2, %3; sub.s32 w3, " #W "3, %3;\n" \
    "abs.s32 t0, w0; abs.s32 t1, w1; abs.s32 t2, w2; abs.s32 t3, w3;\n"                                \
    "add.s32 u0, t0, -1; add.s32 u1, t1, -1; add.s32 u2, t2, -1; add.s32 u3, t3, -1;\n"                \
    "lop3.b32 t0, t0, u0, nm, 0xE0; lop3.b32 t1, t1, u1, nm, 0xE0; lop3.b32 t2, t2, u2, nm, 0xE0; lop3.b32 t3, t3, u3, nm, 0xE0;\n" \
    "dp4a.u32.u32 t0, t0, on, zr; dp4a.u32.u32 t1, t1, on, zr; dp4a.u32.u32 t2, t2, on, zr; dp4a.u32.u32 t3, t3, on, zr;\n" \
    "mul.lo.u32 t0, t0, 32; mul.lo.u32 t2, t2, 32;\n"                                                  \
    "shr.u32 w0, w0, t0; shr.u32 w2, w2, t2;\n"                                                        \
    "setp.eq.u32 p1, t1, 0; setp.eq.u32 p3, t3, 0;\n"                                                  \
    "lop3.b32 A, A, w0, w2, 0x96; @p1 xor.b32 A, A, w1; @p3 xor.b32 A, A, w3;\n"

__device__ __forceinline__ uint32_t scan_dpw(uint32_t addr, uint32_t T, uint32_t h)
{
    uint32_t A;
    asm volatile("{\n"
        ".reg .pred q, p1, p3;\n"
        ".reg .b32 a0, a1, a2, a3, b0, b1, b2, b3, ad, od, cnt, A, nm, on, zr, w0, w1, w2, w3, t0, t1, t2, t3, u0, u1, u2, u3;\n"
        "mov.u32 ad, %1; mov.u32 cnt, %2; mov.u32 A, 0; mov.u32 nm, 0xFFEFFBFE; mov.u32 on, 0x01010101; mov.u32 zr, 0;\n"
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad];\n"
        "and.b32 od, cnt, 1;\n"
        "setp.eq.u32 q, od, 0;\n"
        "@q bra DPW_EVEN;\n"
        ROSEN_DPW_CHUNK(a)
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad+16];\n"
        "add.u32 ad, ad, 16; sub.u32 cnt, cnt, 1;\n"
        "DPW_EVEN:\n"
        "setp.eq.u32 q, cnt, 0;\n"
        "@q bra DPW_DONE;\n"
        "DPW_LOOP:\n"
        "ld.shared.v4.b32 {b0, b1, b2, b3}, [ad+16];\n"
        ROSEN_DPW_CHUNK(a)
        "ld.shared.v4.b32 {a0, a1, a2, a3}, [ad+32];\n"
        ROSEN_DPW_CHUNK(b)
        "add.u32 ad, ad, 32; sub.u32 cnt, cnt, 2;\n"
        "setp.ne.u32 q, cnt, 0;\n"
        "@q bra DPW_LOOP;\n"
        "DPW_DONE:\n"
        "mov.u32 %0, A;\n"
        "}\n"
        : "=r"(A)
        : "r"(addr), "r"(T), "r"(h)
        : "memory");
    return A;
}

__device__ __forceinline__ uint4 lds128(uint32_t a) { uint4 v; asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds32(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts128(uint32_t a, uint32_t v) { asm volatile("st.shared.v4.u32 [%0], {%1, %2, %2, %2};" :: "r"(a), "r"(v), "r"(0u) : "memory"); }

// MODE 0: N <= 64, 8-bit fields, lnW from an m histogram; MODE 3: the same for N = 0 (mod 4), without the per-step s < N test. MODE 1: 64 < N <= 128, 8-bit fields, lnW as a running fp64 sum in
// step order (lnW crosses 128 there, where the oracle's step-by-step sum rounds every ln 5 it adds the same way -- a systematic
// 6e-13 relative to the histogram's more accurate value; following the oracle's order keeps the ensemble sums within 1e-13).
// MODE 2 ("wide"): 128 < N <= 512, 10-bit fields, running sum.
template <int MODE, bool DIGEST, bool TRAJ>
__global__ void __launch_bounds__(256) lattice_dp_kernel(const LatticeParams p)
{
    constexpr bool WIDE = MODE == 2, RUNSUM = MODE == 1 || MODE == 2, FULL4 = MODE == 3, SHORT = MODE == 0 || MODE == 3;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    DpTables* tab = reinterpret_cast<DpTables*>(smem_raw);
    Partial* scratch = reinterpret_cast<Partial*>(smem_raw + sizeof(DpTables));
    uint32_t* chains = reinterpret_cast<uint32_t*>(smem_raw + sizeof(DpTables) + 8 * sizeof(Partial));

    constexpr int B = WIDE ? 10 : 8;                         // field width; bias 2^(B-1)
    constexpr uint32_t kFieldMask = (1u << B) - 1u;
    constexpr int kBias = 1 << (B - 1);
    constexpr uint32_t kOrigin = (uint32_t)kBias | ((uint32_t)kBias << B) | ((uint32_t)kBias << (2 * B));
    const int N = p.N;
    const int half4 = half4_of(N), stride = stride_of(N);
    uint32_t* ev = chains + (size_t)threadIdx.x * stride;   // monomers 0,2,4,...
    uint32_t* od = ev + half4;                              // monomers 1,3,5,...
    uint32_t lut_addr = (uint32_t)__cvta_generic_to_shared(tab->lut);
    uint32_t delta_addr = (uint32_t)__cvta_generic_to_shared(tab->delta);
    const uint32_t ev_addr = (uint32_t)__cvta_generic_to_shared(ev);
    const uint32_t od_addr = ev_addr + (uint32_t)half4 * 4u;
    // Opaque copies: otherwise the compiler re-derives the shared-window addresses and the three byte selectors of the
    // coordinate sums with uniform-datapath instructions in every step (7 issue slots per step in the round-1 SASS).
    if (SHORT) asm volatile("" : "+r"(lut_addr), "+r"(delta_addr));      // (measured: helps N <= 64, costs 10 % at N = 128)

    build_dp_tables<B>(tab);
    __syncthreads();

    const uint32_t per_thread = p.chunk / blockDim.x;
    // the byte selectors of the coordinate sums come from memory so that they live in registers (as immediates they are
    // re-materialised by three uniform moves in every step)
    const uint32_t minus1 = SHORT ? (uint32_t)tab->delta[1] : 0xFFFFFFFFu;      // delta of -x = -1
    const int sel_y = SHORT ? tab->delta[6] : 0x100, sel_z = SHORT ? tab->delta[7] : 0x10000, sel_x = sel_y >> 8;

    __shared__ uint32_t vb_ticket;
    for (;;) {
        if (threadIdx.x == 0) vb_ticket = atomicAdd(p.vb_counter, 1u);    // dynamic draw: no tail of idle blocks
        __syncthreads();
        const uint32_t vb = vb_ticket;      // every thread reads it before the barriers inside block_reduce_store
        if (vb >= p.n_vblocks) break;
        Partial acc = partial_zero();
        for (uint32_t it = 0; it < per_thread; ++it) {
            const uint64_t idx = (uint64_t)vb * p.chunk + (uint64_t)it * blockDim.x + threadIdx.x;
            const bool active = idx < p.n_chains;
            if (TRAJ) { if (!__any_sync(0xffffffffu, active)) break; }    // the conformation store below is warp-cooperative:
            else if (!active) break;                                     // lanes past the end grow a chain nobody keeps
            const uint64_t chain = p.chain_offset + idx;
            const uint32_t c_lo = (uint32_t)chain, c_hi = (uint32_t)(chain >> 32);

            // L0. No clearing pass: the first key of every 4-key chunk is stored as {key, 0, 0, 0}, so a scan
            // never sees a key of the previous chain (0 is not a neighbour of any head: every byte of h is >= 1, so
            // |0 - h| >= 0x010101 has at least two nonzero bytes).
            uint32_t h = kOrigin;
            sts128(ev_addr, h);
            int sx = 0, sy = 0, sz = 0, s2 = 0;
            uint32_t hist = 0, dead = 0;     // dead = step of the first m = 0 (0: alive)
            double lnW_w = 0.0;             // RUNSUM: running sum in step order
            uint64_t dg = 0xCBF29CE484222325ull;
            uint8_t* mrow = TRAJ && active && p.out.m_seq ? p.out.m_seq + idx * (uint64_t)(N - 1) : nullptr;

#pragma unroll 2
            for (int q = 0; 4 * q < N; ++q) {
                uint32_t w[4];
                philox4x32_10(c_lo, c_hi, (uint32_t)q, 0u, p.rk, w);   // L1
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int s = 4 * q + k;
                    if (FULL4) { if (k == 0 && q == 0) continue; }            // N = 0 (mod 4): every block serves four steps, but s = 0
                    else if (s == 0 || s >= N) continue;

                    // L2
                    uint32_t A = 0;
                    const uint32_t T = (uint32_t)(((s >> 1) + 3) >> 2);
                    if (T != 0u) A = WIDE ? scan_dpw((k & 1) ? od_addr : ev_addr, T, h) : scan_dp((k & 1) ? od_addr : ev_addr, T, h, minus1);
                    uint32_t li;                                              // 16 * (b0,b1,bB,bB+1,b2B,b2B+1)
                    if (WIDE) { const uint32_t x = A & 0x00300C03u; li = ((x | (x >> 8) | (x >> 16)) & 0x3Fu) << 4; }
                    else li = (((A & 0x00030303u) * 0x00010410u) >> 12) & 0x3F0u;
                    const uint4 le = lds128(lut_addr + li);
                    const uint32_t m = le.w;

                    // L3
                    if (RUNSUM) lnW_w += tab->ln_m[m]; else hist += le.z;
                    if (TRAJ && mrow) mrow[s - 1] = dead == 0u ? (uint8_t)m : (uint8_t)0;

                    // L4
                    const uint32_t sel = __umulhi(w[k], m);
                    const uint32_t d4 = __byte_perm(le.x, le.y, sel) & 0xFFu;   // 4 * direction
                    if (DIGEST) { if (dead == 0u) dg = digest_fold(dg, m, m ? (d4 >> 2) : 0xFFu); }
                    dead = (m == 0u && dead == 0u) ? (uint32_t)s : dead;
                    h += lds32(delta_addr + d4);
                    const uint32_t slot = ((k & 1) ? od_addr : ev_addr) + 4u * (uint32_t)(s >> 1);
                    if (((s >> 1) & 3) == 0) sts128(slot, h); else sts32(slot, h);

                    // L5: signed bytes of r_s; |r|^2 and the three coordinate sums as byte dot products
                    if (WIDE) {
                        const int hx = (int)(h & kFieldMask) - kBias, hy = (int)((h >> B) & kFieldMask) - kBias,
                                  hz = (int)(h >> (2 * B)) - kBias;
                        sx += hx; sy += hy; sz += hz; s2 += hx * hx + hy * hy + hz * hz;
                    } else {
                        const int sg = (int)(h ^ kOrigin);
                        s2 = __dp4a(sg, sg, s2);
                        sx = __dp4a(sg, sel_x, sx); sy = __dp4a(sg, sel_y, sy); sz = __dp4a(sg, sel_z, sz);
                    }
                }
            }

            const bool alive = dead == 0u;
            const uint32_t steps = alive ? (uint32_t)(N - 1) : dead;     // attempted steps
            double lnW = tab->ln_m[6];
            lnW += (double)(hist & 255u) * tab->ln_m[2];
            lnW += (double)((hist >> 8) & 255u) * tab->ln_m[3];
            lnW += (double)((hist >> 16) & 255u) * tab->ln_m[4];
            lnW += (double)(hist >> 24) * tab->ln_m[5];
            if (RUNSUM) lnW = lnW_w;
            if (!alive) lnW = -CUDART_INF;
            double ree2 = 0.0, rg2 = 0.0;
            if (alive) {
                const int hx = (int)(h & kFieldMask) - kBias, hy = (int)((h >> B) & kFieldMask) - kBias,
                          hz = (int)(h >> (2 * B)) - kBias;
                ree2 = (double)(hx * hx + hy * hy + hz * hz);
                const long long num = (long long)N * s2 - ((long long)sx * sx + (long long)sy * sy + (long long)sz * sz);
                rg2 = (double)num / ((double)N * (double)N);
            }
            const double wgt = alive ? exp(lnW - p.ln_shift) : 0.0;
            if (!TRAJ || active) {
                acc.sum_w += wgt; acc.sum_w_ree2 += wgt * ree2; acc.sum_w_rg2 += wgt * rg2; acc.sum_w2 += wgt * wgt;
                acc.n_dead += alive ? 0u : 1u; acc.n_steps += steps;
                if (DIGEST) { acc.digest_xor ^= dg; acc.digest_sum += dg; }

                if (p.out.lnW) p.out.lnW[idx] = lnW;
                if (p.out.alive) p.out.alive[idx] = alive ? 1 : 0;
                if (p.out.ree2) p.out.ree2[idx] = ree2;
                if (p.out.rg2) p.out.rg2[idx] = rg2;
                if (DIGEST && p.out.digest) p.out.digest[idx] = dg;
            }
            if (TRAJ && p.out.conf) {
                // D1: the warp stores its 32 chains one after the other, consecutive lanes writing consecutive int32 of the
                // chain's [N][3] row block (128 contiguous bytes per instruction); zeros from the death step on.
                __syncwarp();
                const int lane = threadIdx.x & 31;
                const int my_placed = active ? (alive ? N : (int)steps) : -1;
                const uint32_t* wbase = chains + (size_t)(threadIdx.x - lane) * stride;
                for (int L = 0; L < 32; ++L) {
                    const int placed = __shfl_sync(0xffffffffu, my_placed, L);
                    if (placed < 0) continue;                                  // warp-uniform
                    const uint32_t* cev = wbase + (size_t)L * stride;
                    const uint32_t* cod = cev + half4;
                    int32_t* c = reinterpret_cast<int32_t*>(p.out.conf) + (idx - lane + L) * (uint64_t)N * 3;
                    for (int e = lane; e < 3 * N; e += 32) {
                        const int i = (int)(((uint32_t)e * 43691u) >> 17), a = e - 3 * i;      // e / 3, e % 3 (e < 98304)
                        const uint32_t v = ((i & 1) ? cod : cev)[i >> 1];
                        c[e] = i < placed ? (int)((v >> (B * a)) & kFieldMask) - kBias : 0;
                    }
                }
                __syncwarp();
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

template <int MODE>
int launch_dp(const LatticeParams& p, cudaStream_t stream, int* grid_out)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    const size_t tb = sizeof(DpTables);
    if (traj) return digest ? launch_kernel(lattice_dp_kernel<MODE, true, true>, tb, p, stream, grid_out)
                            : launch_kernel(lattice_dp_kernel<MODE, false, true>, tb, p, stream, grid_out);
    return digest ? launch_kernel(lattice_dp_kernel<MODE, true, false>, tb, p, stream, grid_out)
                  : launch_kernel(lattice_dp_kernel<MODE, false, false>, tb, p, stream, grid_out);
}

}  // namespace

int launch_lattice(const LatticeParams& p, cudaStream_t stream, const char** kernel_name, int* grid_out)
{
    const bool digest = p.out.digest != nullptr;
    const bool traj = p.out.m_seq != nullptr || p.out.conf != nullptr;
    if (p.N <= 128) {   // every scanned difference |dx|,|dy|,|dz| <= s-1-j <= 126 fits a signed byte: byte-dot-product scan
        *kernel_name = traj ? (digest ? "lattice_dp_kernel<digest,traj>" : "lattice_dp_kernel<traj>")
                            : (digest ? "lattice_dp_kernel<digest>" : "lattice_dp_kernel");
        if (p.N <= 64) return (p.N & 3) == 0 ? launch_dp<3>(p, stream, grid_out) : launch_dp<0>(p, stream, grid_out);
        return launch_dp<1>(p, stream, grid_out);
    }
    // 10-bit fields (|d| <= 510 < 2^9, 128 < N <= 512): power-of-two test + byte-sum scan
    *kernel_name = traj ? (digest ? "lattice_dp_kernel<wide,digest,traj>" : "lattice_dp_kernel<wide,traj>")
                        : (digest ? "lattice_dp_kernel<wide,digest>" : "lattice_dp_kernel<wide>");
    return launch_dp<2>(p, stream, grid_out);
}

}  // namespace rosen
