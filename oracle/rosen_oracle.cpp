// rosen_oracle.cpp -- TEST INFRASTRUCTURE. Plain, slow, single-threaded CPU oracle for the
// Rosenbluth chain-generation hot path of arXiv 1704.04381 (Guo & Baulin, CPC 2017).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this library. It shares no code, header, table or constant generator with the CUDA path
// (paper_1704_04381_b200/csrc); both sides restate DESIGN.md section 3 ("numeric specification")
// independently. Every function follows the paper's algorithm step by step, in its order and
// notation; no blocking, fusion or pruning (the full j = 0..s-2 scans of Alg. 1 / Alg. 2 are kept).
//
// Citations are PAPER.md line numbers (= /root/reference/PAPER.md) plus section / algorithm.
// Readings A1..A15 of the garbled / ambiguous passages are listed in DESIGN.md section 4.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"):
//   philox4x32_10          : Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt)
//   lattice free-site count: sum over ALL enumerated SAWs of 1/W == P_alive exactly (saw_enum.cpp)
//   lattice grower+weights : mean(W) -> c_n, W-weighted <Ree2>,<Rg2> -> exact enumeration means
//   real-space grower      : N=3 closed forms (free fraction 3/4, <Ree2>=2.5, <Rg2>=0.5),
//                            sigma=0 freely-jointed chain (<Ree2>=(N-1)b^2, <Rg2>=b^2(N^2-1)/(6N))
//   unit-sphere direction  : against fp64 libm cos/sin of the exact angle; |u|=1; moments
//   parity unpinned        : none of the exported functions; real-space N>=4 with sigma>0 has no
//                            closed form, it is covered by the invariants (bond length, no overlap)
//                            and by the two special cases above only.
//
// Build: g++ -O2 -ffp-contract=off -shared -fPIC (see oracle/build.py). fp32 arithmetic of the
// real-space path is written operation by operation with std::fmaf where DESIGN.md says "fma".

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

extern "C" {

// ---------------------------------------------------------------------------------------------
// Result layouts (host memory; mirrors include/rosen.h field by field but is declared here
// independently -- the oracle does not include the product header).
// ---------------------------------------------------------------------------------------------
struct oracle_summary {
    uint64_t n_chains, n_dead, n_steps_attempted;
    double   ln_shift;                                   // L
    double   sum_w, sum_w_ree2, sum_w_rg2, sum_w2;       // w = exp(lnW - L); dead chains add 0
    double   mean_ree2, mean_rg2, attrition, ln_mean_W;  // derived
    uint64_t digest_xor, digest_sum;
};

struct oracle_outputs {     // every pointer optional (NULL = not written), HOST memory
    double*   lnW;          // [n_chains]   -inf for dead chains
    uint8_t*  alive;        // [n_chains]
    uint8_t*  m_seq;        // [n_chains][N-1]  0 from the death step on
    uint64_t* digest;       // [n_chains]
    void*     conf;         // [n_chains][N][3] int32 (lattice) / float (real space); 0 after death
    double*   ree2;         // [n_chains]
    double*   rg2;          // [n_chains]
};

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11). BASELINE north_star replaces the paper's
// cuRAND generator (sec. 3.2) by this counter-based one; DESIGN.md 3.1.
// ---------------------------------------------------------------------------------------------
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }   // Weyl key schedule
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Word used by growth step s of chain `chain` for the uniform choice among free trials
// (DESIGN.md 3.1 / reading A9): block counter (chain_lo, chain_hi, s>>2, 0), word s&3.
static uint32_t selection_word(uint64_t seed, uint64_t chain, uint32_t s)
{
    const uint32_t ctr[4] = { (uint32_t)chain, (uint32_t)(chain >> 32), s >> 2, 0u };
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[s & 3u];
}

// Per-chain digest of the decisions: FNV-1a style fold of one 32-bit token per
// attempted step, token = m_s | choice_s << 8, choice = 0xFF on the death step.
static inline uint64_t digest_init() { return 0xCBF29CE484222325ull; }
static inline uint64_t digest_fold(uint64_t h, uint32_t m, uint32_t choice)
{
    return (h ^ (uint64_t)(m | (choice << 8))) * 0x100000001B3ull;
}

// Neumaier compensated accumulator for the ensemble sums (so that the oracle's own rounding
// does not eat the 1e-12 parity tolerance).
struct Comp {
    double s = 0.0, c = 0.0;
    void add(double x) {
        const double t = s + x;
        if (std::fabs(s) >= std::fabs(x)) c += (s - t) + x; else c += (x - t) + s;
        s = t;
    }
    double value() const { return s + c; }
};

// ---------------------------------------------------------------------------------------------
// Lattice: the six trial sites, in the fixed order +x,-x,+y,-y,+z,-z.
// ---------------------------------------------------------------------------------------------
static const int32_t E[6][3] = { {1,0,0}, {-1,0,0}, {0,1,0}, {0,-1,0}, {0,0,1}, {0,0,-1} };

// Free-site list at a growth step (PAPER.md:126-149 Alg. 1 lines 9-23 overlap loop; :157-176
// lines 24-34 neighbour count; readings A2, A3): trial d is free iff r[s-1]+e_d differs from
// every earlier monomer r[j], j = 0..s-2 (the scan also covers j = s-1, which can never match).
// r = s placed monomers [s][3]. Returns m = number of free trials, free_dirs[0..m) ascending.
int32_t oracle_lattice_free_dirs(const int32_t* r, int32_t s, int32_t free_dirs[6])
{
    int32_t m = 0;
    for (int d = 0; d < 6; ++d) {
        const int32_t tx = r[3 * (s - 1) + 0] + E[d][0];
        const int32_t ty = r[3 * (s - 1) + 1] + E[d][1];
        const int32_t tz = r[3 * (s - 1) + 2] + E[d][2];
        bool overlap = false;
        for (int j = 0; j < s - 1; ++j)                                   // Alg. 1 line 13
            if (r[3 * j] == tx && r[3 * j + 1] == ty && r[3 * j + 2] == tz) overlap = true;
        if (!overlap) free_dirs[m++] = d;
    }
    return m;
}

static void finish_summary(oracle_summary* S, uint64_t n_chains, uint64_t n_dead, uint64_t n_steps,
                           double L, const Comp& sw, const Comp& swr, const Comp& swg, const Comp& sw2,
                           uint64_t dx, uint64_t ds)
{
    if (!S) return;
    S->n_chains = n_chains; S->n_dead = n_dead; S->n_steps_attempted = n_steps; S->ln_shift = L;
    S->sum_w = sw.value(); S->sum_w_ree2 = swr.value(); S->sum_w_rg2 = swg.value(); S->sum_w2 = sw2.value();
    S->mean_ree2 = S->sum_w_ree2 / S->sum_w;                              // Eq. 2
    S->mean_rg2  = S->sum_w_rg2 / S->sum_w;
    S->attrition = (double)n_dead / (double)n_chains;
    S->ln_mean_W = L + std::log(S->sum_w / (double)n_chains);             // Eq. 6
    S->digest_xor = dx; S->digest_sum = ds;
}

// Ensemble sums, Eq. 2 and Eq. 6 (:362), over the stored per-chain results in chain order.
// `long_chain` (lattice N > 512, real space N > 2048, reading A18): the shift is the largest lnW of the
// run instead of the fixed bound L_fixed, because exp(lnW - L_fixed) underflows fp64 for chains of 10^4 monomers.
// Any L cancels in the ratios of Eq. 2 and is added back in Eq. 6; with no chain alive L = 0 and the means are 0/0.
struct ChainResult { double lnW, ree2, rg2; bool alive; };

static void ensemble(oracle_summary* S, const std::vector<ChainResult>& res, bool long_chain, double L_fixed,
                     uint64_t n_steps, uint64_t dx, uint64_t ds)
{
    double L = L_fixed;
    if (long_chain) {
        bool any = false;
        for (const ChainResult& c : res) if (c.alive && (!any || c.lnW > L)) { L = c.lnW; any = true; }
        if (!any) L = 0.0;
    }
    Comp sw, swr, swg, sw2;
    uint64_t n_dead = 0;
    for (const ChainResult& c : res) {
        const double w = c.alive ? std::exp(c.lnW - L) : 0.0;
        sw.add(w); swr.add(w * c.ree2); swg.add(w * c.rg2); sw2.add(w * w);
        if (!c.alive) ++n_dead;
    }
    finish_summary(S, (uint64_t)res.size(), n_dead, n_steps, L, sw, swr, swg, sw2, dx, ds);
}

// Cubic-lattice Rosenbluth generation, PAPER.md:100-179 (Alg. 1), Eq. 3 (:58), sec. 3.3.2.
// Returns 0, or -1 on invalid arguments.
int oracle_lattice_generate(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                            const oracle_outputs* out, oracle_summary* summary)
{
    if (N < 2 || n_chains == 0) return -1;
    const double L = std::log(6.0) + (double)(N - 2) * std::log(5.0);     // max possible lnW (fixed shift, N <= 512)
    std::vector<int32_t> r((size_t)N * 3);
    std::vector<ChainResult> res;
    res.reserve(n_chains);
    uint64_t n_steps = 0, dxor = 0, dsum = 0;

    for (uint64_t i = 0; i < n_chains; ++i) {
        const uint64_t chain = chain_offset + i;
        std::fill(r.begin(), r.end(), 0);                                 // Pos[0] <- 0, :119
        double lnW = 0.0;                                                 // W = 1
        bool alive = true;
        uint64_t h = digest_init();
        uint8_t* mrow = (out && out->m_seq) ? out->m_seq + i * (size_t)(N - 1) : nullptr;
        if (mrow) std::memset(mrow, 0, (size_t)(N - 1));

        for (int32_t s = 1; s <= N - 1; ++s) {                            // Alg. 1 line 4
            int32_t free_dirs[6];
            const int32_t m = oracle_lattice_free_dirs(r.data(), s, free_dirs);
            ++n_steps;
            if (mrow) mrow[s - 1] = (uint8_t)m;
            if (m == 0) {                                                 // dead end, :98; reading A6
                alive = false; h = digest_fold(h, 0, 0xFF);
                for (int32_t q = s; q < N; ++q) r[3*q] = r[3*q+1] = r[3*q+2] = 0;
                break;
            }
            lnW += std::log((double)m);                                   // W *= 1/p_i = m, Eq. 3
            const uint32_t u = selection_word(seed, chain, (uint32_t)s);
            const uint32_t sel = (uint32_t)(((uint64_t)u * (uint64_t)m) >> 32);   // reading A7
            const int32_t d = free_dirs[sel];
            r[3*s+0] = r[3*(s-1)+0] + E[d][0];                            // Alg. 1 line 19
            r[3*s+1] = r[3*(s-1)+1] + E[d][1];
            r[3*s+2] = r[3*(s-1)+2] + E[d][2];
            h = digest_fold(h, (uint32_t)m, (uint32_t)d);
        }

        // observables (sec. 4.1; Rg2 from north_star): integers until the divide
        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            int64_t sx = 0, sy = 0, sz = 0, s2 = 0;
            for (int32_t q = 0; q < N; ++q) {
                const int64_t x = r[3*q], y = r[3*q+1], z = r[3*q+2];
                sx += x; sy += y; sz += z; s2 += x*x + y*y + z*z;
            }
            const int64_t ex = r[3*(N-1)] - r[0], ey = r[3*(N-1)+1] - r[1], ez = r[3*(N-1)+2] - r[2];
            ree2 = (double)(ex*ex + ey*ey + ez*ez);
            rg2  = (double)((int64_t)N * s2 - (sx*sx + sy*sy + sz*sz)) / ((double)N * (double)N);
        } else {
            lnW = -std::numeric_limits<double>::infinity();
        }
        res.push_back(ChainResult{lnW, ree2, rg2, alive});
        dxor ^= h; dsum += h;

        if (out) {
            if (out->lnW) out->lnW[i] = lnW;
            if (out->alive) out->alive[i] = alive ? 1 : 0;
            if (out->digest) out->digest[i] = h;
            if (out->ree2) out->ree2[i] = ree2;
            if (out->rg2) out->rg2[i] = rg2;
            if (out->conf) std::memcpy((int32_t*)out->conf + i * (size_t)N * 3, r.data(), (size_t)N * 3 * sizeof(int32_t));
        }
    }
    ensemble(summary, res, N > 512, L, n_steps, dxor, dsum);
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Real space (PAPER.md:185-187 sec. 3.3.3, :202-262 Alg. 2).
// ---------------------------------------------------------------------------------------------

// "rngonsphere" (Alg. 2 line 10), re-specified on two Philox words so that it is
// reproducible to the bit on any IEEE-754 machine (reading A10): only
// + - * fma sqrt, all correctly rounded; no libm trigonometry.
void oracle_direction(uint32_t wz, uint32_t wphi, float u[3])
{
    // z uniform on the 2^23 midpoints of (-1,1); exact in fp32
    const float z = std::fmaf((float)(2u * (wz >> 9) + 1u), 0x1p-23f, -1.0f);
    // azimuth: 24 bits = 3 octant bits + 21 fraction bits; odd octants are mirrored
    const uint32_t a = wphi >> 8;
    const uint32_t oct = a >> 21;
    const uint32_t f = a & 0x1FFFFFu;
    const uint32_t g = (oct & 1u) ? (0x1FFFFFu - f) : f;
    const float x = (float)(2u * g + 1u) * 0x1.921fb6p-23f;             // (2g+1) * fl(pi/4 * 2^-22)
    const float x2 = x * x;
    // sin x, cos x on (0, pi/4): Taylor polynomials, coefficients = fp32-nearest of +-1/n!
    float p = std::fmaf(x2, 0x1.71de3ap-19f, -0x1.a01a02p-13f);          // 1/9!, -1/7!
    p = std::fmaf(x2, p, 0x1.111112p-7f);                                // 1/5!
    p = std::fmaf(x2, p, -0x1.555556p-3f);                               // -1/3!
    p = p * x2;
    const float sn = std::fmaf(x, p, x);
    float q = std::fmaf(x2, -0x1.27e4fcp-22f, 0x1.a01a02p-16f);          // -1/10!, 1/8!
    q = std::fmaf(x2, q, -0x1.6c16c2p-10f);                              // -1/6!
    q = std::fmaf(x2, q, 0x1.555556p-5f);                                // 1/4!
    q = std::fmaf(x2, q, -0.5f);                                         // -1/2!
    const float cs = std::fmaf(x2, q, 1.0f);
    // octant table (cos phi, sin phi): 0:(c,s) 1:(s,c) 2:(-s,c) 3:(-c,s) 4:(-c,-s) 5:(-s,-c) 6:(s,-c) 7:(c,-s)
    const bool swap = (((oct + 1u) >> 1) & 1u) != 0;
    float cx = swap ? sn : cs;
    float sy = swap ? cs : sn;
    if (oct >= 2u && oct <= 5u) cx = -cx;
    if (oct >= 4u) sy = -sy;
    const float rho = std::sqrt(std::fmaf(-z, z, 1.0f));
    u[0] = rho * cx; u[1] = rho * sy; u[2] = z;
}

// Words of trial t at growth step s (DESIGN.md 3.1 / reading A9): block counter
// (chain_lo, chain_hi, s, 1 + (t>>1)); even t takes words (0,1), odd t words (2,3).
static void trial_words(uint64_t seed, uint64_t chain, uint32_t s, uint32_t t, uint32_t* wz, uint32_t* wphi)
{
    const uint32_t ctr[4] = { (uint32_t)chain, (uint32_t)(chain >> 32), s, 1u + (t >> 1) };
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    *wz = out[2 * (t & 1u)]; *wphi = out[2 * (t & 1u) + 1];
}

int oracle_realspace_generate(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                              uint64_t seed, uint64_t chain_offset,
                              const oracle_outputs* out, oracle_summary* summary)
{
    if (N < 2 || n_chains == 0 || k_trials < 1 || k_trials > 255) return -1;
    if (!(bond_len > 0.0f) || !(sigma >= 0.0f) || !std::isfinite(bond_len) || !std::isfinite(sigma)) return -1;
    const int32_t k = k_trials;
    const float b = bond_len;
    const float sigma2 = sigma * sigma;                                   // rounded once to fp32
    const double L = (double)(N - 1) * std::log((double)k);
    std::vector<float> r((size_t)N * 3);
    std::vector<float> trial((size_t)k * 3);
    std::vector<int32_t> free_t((size_t)k);
    std::vector<ChainResult> res;
    res.reserve(n_chains);
    uint64_t n_steps = 0, dxor = 0, dsum = 0;

    for (uint64_t i = 0; i < n_chains; ++i) {
        const uint64_t chain = chain_offset + i;
        std::fill(r.begin(), r.end(), 0.0f);                              // Pos[0] <- 0, :216
        double lnW = 0.0;
        bool alive = true;
        uint64_t h = digest_init();
        uint8_t* mrow = (out && out->m_seq) ? out->m_seq + i * (size_t)(N - 1) : nullptr;
        if (mrow) std::memset(mrow, 0, (size_t)(N - 1));

        for (int32_t s = 1; s <= N - 1; ++s) {                            // Alg. 2 line 4
            const float hx = r[3*(s-1)], hy = r[3*(s-1)+1], hz = r[3*(s-1)+2];
            int32_t m = 0;
            for (int32_t t = 0; t < k; ++t) {                             // Alg. 2 line 9, ptMax = k
                uint32_t wz, wphi; float u[3];
                trial_words(seed, chain, (uint32_t)s, (uint32_t)t, &wz, &wphi);
                oracle_direction(wz, wphi, u);                            // rngonsphere, line 10
                const float tx = std::fmaf(b, u[0], hx);                  // line 11
                const float ty = std::fmaf(b, u[1], hy);
                const float tz = std::fmaf(b, u[2], hz);
                trial[3*t] = tx; trial[3*t+1] = ty; trial[3*t+2] = tz;
                bool overlap = false;
                for (int32_t j = 0; j < s - 1; ++j) {                     // line 13, half-open (A2)
                    const float dx = r[3*j] - tx, dy = r[3*j+1] - ty, dz = r[3*j+2] - tz;
                    const float d2 = std::fmaf(dz, dz, std::fmaf(dy, dy, dx * dx));   // "distance", :235
                    if (d2 < sigma2) overlap = true;                      // strict <, sigma (A11)
                }
                if (!overlap) free_t[m++] = t;                            // counts TRIALS (A5)
            }
            ++n_steps;
            if (mrow) mrow[s - 1] = (uint8_t)m;
            if (m == 0) {                                                 // N_allowed = 0, :187; A6
                alive = false; h = digest_fold(h, 0, 0xFF);
                for (int32_t q = s; q < N; ++q) r[3*q] = r[3*q+1] = r[3*q+2] = 0.0f;
                break;
            }
            lnW += std::log((double)m);                                   // W *= N_allowed (A4)
            const uint32_t u32 = selection_word(seed, chain, (uint32_t)s);
            const uint32_t sel = (uint32_t)(((uint64_t)u32 * (uint64_t)m) >> 32);
            const int32_t t = free_t[sel];
            r[3*s] = trial[3*t]; r[3*s+1] = trial[3*t+1]; r[3*s+2] = trial[3*t+2];   // line 21
            h = digest_fold(h, (uint32_t)m, (uint32_t)t);
        }

        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            double cx = 0.0, cy = 0.0, cz = 0.0;
            for (int32_t q = 0; q < N; ++q) { cx += (double)r[3*q]; cy += (double)r[3*q+1]; cz += (double)r[3*q+2]; }
            cx /= (double)N; cy /= (double)N; cz /= (double)N;
            double acc = 0.0;
            for (int32_t q = 0; q < N; ++q) {
                const double ax = (double)r[3*q] - cx, ay = (double)r[3*q+1] - cy, az = (double)r[3*q+2] - cz;
                acc += ax*ax + ay*ay + az*az;
            }
            rg2 = acc / (double)N;
            const double ex = (double)r[3*(N-1)] - (double)r[0], ey = (double)r[3*(N-1)+1] - (double)r[1],
                         ez = (double)r[3*(N-1)+2] - (double)r[2];
            ree2 = ex*ex + ey*ey + ez*ez;
        } else {
            lnW = -std::numeric_limits<double>::infinity();
        }
        res.push_back(ChainResult{lnW, ree2, rg2, alive});
        dxor ^= h; dsum += h;

        if (out) {
            if (out->lnW) out->lnW[i] = lnW;
            if (out->alive) out->alive[i] = alive ? 1 : 0;
            if (out->digest) out->digest[i] = h;
            if (out->ree2) out->ree2[i] = ree2;
            if (out->rg2) out->rg2[i] = rg2;
            if (out->conf) std::memcpy((float*)out->conf + i * (size_t)N * 3, r.data(), (size_t)N * 3 * sizeof(float));
        }
    }
    ensemble(summary, res, N > 2048, L, n_steps, dxor, dsum);
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Other trial sets and Boltzmann-weighted trials (readings A19-A21).
//
//   * z = 26: "randomly chosen within all z = 26 possible lattice space" (sec. 3.3.2): the trial sites
//     are the 26 sites (dx,dy,dz) in {-1,0,1}^3 \ {0} around r_{s-1}, in the order i = (dx+1) + 3(dy+1) + 9(dz+1)
//     (i = 13, the centre, skipped); self-avoidance is site exclusion only.
//   * Boltzmann weights (Eq. 1-2: configurations enter with exp[-beta U] / P_s): U = -eps per
//     non-bonded contact (lattice: an earlier monomer on one of the z neighbour sites of the new monomer; real space:
//     an earlier monomer closer than lambda sigma), so a free trial t that would make c_t contacts carries the factor
//     q^c_t, q = exp(beta eps); the step's Rosenbluth factor is W_s = sum_t q^c_t and trial t is taken with
//     probability q^c_t / W_s. beta eps = 0 gives back W_s = m_s and the uniform choice of Alg. 1 / Alg. 2.
//   * The factors are FIXED-POINT integers Q[c] = round(q^c 2^16) (q^c by repeated fp64 multiplication), so W_s and
//     the cumulative sums of the choice are exact integers, independent of summation order; the choice is the first
//     trial, in trial order, whose cumulative sum exceeds floor(u_s W_s / 2^32). lnW += log(W_s 2^-16) in fp64.
// ---------------------------------------------------------------------------------------------
void oracle_model_table(double beta_eps, uint64_t Q[32])
{
    const double q = std::exp(beta_eps);
    double p = 1.0;
    for (int c = 0; c < 32; ++c) { Q[c] = (uint64_t)std::llround(p * 65536.0); p *= q; }
}

static void model_dir(int32_t z, int32_t d, int32_t e[3])
{
    if (z == 6) { e[0] = E[d][0]; e[1] = E[d][1]; e[2] = E[d][2]; return; }
    const int32_t i = d < 13 ? d : d + 1;
    e[0] = i % 3 - 1; e[1] = (i / 3) % 3 - 1; e[2] = i / 9 - 1;
}

static bool model_neighbours(int32_t z, const int32_t a[3], const int32_t b[3])
{
    const int32_t dx = std::abs(a[0] - b[0]), dy = std::abs(a[1] - b[1]), dz = std::abs(a[2] - b[2]);
    if (dx + dy + dz == 0) return false;
    return z == 6 ? dx + dy + dz == 1 : (dx <= 1 && dy <= 1 && dz <= 1);
}

// One growth step of the lattice model: r = s placed monomers [s][3]; for every trial d (order above) w[d] = 0 if the
// site r[s-1] + e_d is occupied by some r[j], j <= s-2, else Q[c_d] with c_d = number of j <= s-2 whose site is a
// z-neighbour of the trial site (the bonded predecessor r[s-1] is not counted). Returns m = number of free trials.
int32_t oracle_lattice_model_step(const int32_t* r, int32_t s, int32_t z, const uint64_t Q[32], uint64_t w[26])
{
    int32_t m = 0;
    for (int32_t d = 0; d < z; ++d) {
        int32_t e[3], t[3];
        model_dir(z, d, e);
        for (int a = 0; a < 3; ++a) t[a] = r[3 * (s - 1) + a] + e[a];
        bool overlap = false;
        int32_t c = 0;
        for (int32_t j = 0; j < s - 1; ++j) {
            if (r[3*j] == t[0] && r[3*j+1] == t[1] && r[3*j+2] == t[2]) overlap = true;
            if (model_neighbours(z, &r[3*j], t)) ++c;
        }
        w[d] = overlap ? 0 : Q[c];
        if (!overlap) ++m;
    }
    return m;
}

// floor(u W / 2^32) for a 32-bit u and W < 2^63, without a 128-bit product
static uint64_t scaled_target(uint32_t u, uint64_t W)
{
    return (W >> 32) * (uint64_t)u + (((W & 0xFFFFFFFFull) * (uint64_t)u) >> 32);
}

// the same routine, exported so that a test can pin it against Python's big integers: (u W) >> 32
uint64_t oracle_scaled_target(uint32_t u, uint64_t W) { return scaled_target(u, W); }

int oracle_lattice_model_generate(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset, int32_t z,
                                  double beta_eps, const oracle_outputs* out, oracle_summary* summary)
{
    if (N < 2 || n_chains == 0 || (z != 6 && z != 26) || !(beta_eps >= 0.0) || !(beta_eps <= 0.85)) return -1;
    uint64_t Q[32];
    oracle_model_table(beta_eps, Q);
    std::vector<int32_t> r((size_t)N * 3);
    std::vector<ChainResult> res;
    res.reserve(n_chains);
    uint64_t n_steps = 0, dxor = 0, dsum = 0;

    for (uint64_t i = 0; i < n_chains; ++i) {
        const uint64_t chain = chain_offset + i;
        std::fill(r.begin(), r.end(), 0);
        double lnW = 0.0;
        bool alive = true;
        uint64_t h = digest_init();
        uint8_t* mrow = (out && out->m_seq) ? out->m_seq + i * (size_t)(N - 1) : nullptr;
        if (mrow) std::memset(mrow, 0, (size_t)(N - 1));

        for (int32_t s = 1; s <= N - 1; ++s) {
            uint64_t w[26];
            const int32_t m = oracle_lattice_model_step(r.data(), s, z, Q, w);
            ++n_steps;
            if (mrow) mrow[s - 1] = (uint8_t)m;
            if (m == 0) {
                alive = false; h = digest_fold(h, 0, 0xFF);
                for (int32_t q = s; q < N; ++q) r[3*q] = r[3*q+1] = r[3*q+2] = 0;
                break;
            }
            uint64_t W = 0;
            for (int32_t d = 0; d < z; ++d) W += w[d];
            lnW += std::log((double)W * 0x1p-16);                          // W_s = sum_t q^c_t
            const uint64_t target = scaled_target(selection_word(seed, chain, (uint32_t)s), W);
            int32_t d = 0;
            uint64_t cum = w[0];
            while (cum <= target) cum += w[++d];                         // first trial whose cumulative sum exceeds the target
            int32_t e[3];
            model_dir(z, d, e);
            for (int a = 0; a < 3; ++a) r[3*s+a] = r[3*(s-1)+a] + e[a];
            h = digest_fold(h, (uint32_t)m, (uint32_t)d);
        }

        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            int64_t sx = 0, sy = 0, sz = 0, s2 = 0;
            for (int32_t q = 0; q < N; ++q) {
                const int64_t x = r[3*q], y = r[3*q+1], zz = r[3*q+2];
                sx += x; sy += y; sz += zz; s2 += x*x + y*y + zz*zz;
            }
            const int64_t ex = r[3*(N-1)], ey = r[3*(N-1)+1], ez = r[3*(N-1)+2];
            ree2 = (double)(ex*ex + ey*ey + ez*ez);
            rg2  = (double)((int64_t)N * s2 - (sx*sx + sy*sy + sz*sz)) / ((double)N * (double)N);
        } else {
            lnW = -std::numeric_limits<double>::infinity();
        }
        res.push_back(ChainResult{lnW, ree2, rg2, alive});
        dxor ^= h; dsum += h;
        if (out) {
            if (out->lnW) out->lnW[i] = lnW;
            if (out->alive) out->alive[i] = alive ? 1 : 0;
            if (out->digest) out->digest[i] = h;
            if (out->ree2) out->ree2[i] = ree2;
            if (out->rg2) out->rg2[i] = rg2;
            if (out->conf) std::memcpy((int32_t*)out->conf + i * (size_t)N * 3, r.data(), (size_t)N * 3 * sizeof(int32_t));
        }
    }
    ensemble(summary, res, true, 0.0, n_steps, dxor, dsum);             // shift = largest lnW of the call (reading A18)
    return 0;
}

// Real space with a square-well attraction: trial t overlaps as in Alg. 2 (d2 < sigma2); a free trial
// carries Q[min(n_t, 31)], n_t = number of earlier monomers j <= s-2 with d2 < well2, well = fl32(lambda sigma),
// well2 = fl32(well well), d2 the same fp32 expression as the overlap test. lambda >= 1.
int oracle_realspace_model_generate(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                                    float lambda, double beta_eps, uint64_t seed, uint64_t chain_offset,
                                    const oracle_outputs* out, oracle_summary* summary)
{
    if (N < 2 || n_chains == 0 || k_trials < 1 || k_trials > 255) return -1;
    if (!(bond_len > 0.0f) || !(sigma >= 0.0f) || !std::isfinite(bond_len) || !std::isfinite(sigma)) return -1;
    if (!(lambda >= 1.0f) || !std::isfinite(lambda) || !(beta_eps >= 0.0) || !(beta_eps <= 0.85)) return -1;
    uint64_t Q[32];
    oracle_model_table(beta_eps, Q);
    const int32_t k = k_trials;
    const float b = bond_len;
    const float sigma2 = sigma * sigma;
    const float well = lambda * sigma;
    const float well2 = well * well;
    std::vector<float> r((size_t)N * 3);
    std::vector<float> trial((size_t)k * 3);
    std::vector<uint64_t> w((size_t)k);
    std::vector<ChainResult> res;
    res.reserve(n_chains);
    uint64_t n_steps = 0, dxor = 0, dsum = 0;

    for (uint64_t i = 0; i < n_chains; ++i) {
        const uint64_t chain = chain_offset + i;
        std::fill(r.begin(), r.end(), 0.0f);
        double lnW = 0.0;
        bool alive = true;
        uint64_t h = digest_init();
        uint8_t* mrow = (out && out->m_seq) ? out->m_seq + i * (size_t)(N - 1) : nullptr;
        if (mrow) std::memset(mrow, 0, (size_t)(N - 1));

        for (int32_t s = 1; s <= N - 1; ++s) {
            const float hx = r[3*(s-1)], hy = r[3*(s-1)+1], hz = r[3*(s-1)+2];
            int32_t m = 0;
            uint64_t W = 0;
            for (int32_t t = 0; t < k; ++t) {
                uint32_t wz, wphi; float u[3];
                trial_words(seed, chain, (uint32_t)s, (uint32_t)t, &wz, &wphi);
                oracle_direction(wz, wphi, u);
                const float tx = std::fmaf(b, u[0], hx), ty = std::fmaf(b, u[1], hy), tz = std::fmaf(b, u[2], hz);
                trial[3*t] = tx; trial[3*t+1] = ty; trial[3*t+2] = tz;
                bool overlap = false;
                int32_t n_well = 0;
                for (int32_t j = 0; j < s - 1; ++j) {
                    const float dx = r[3*j] - tx, dy = r[3*j+1] - ty, dz = r[3*j+2] - tz;
                    const float d2 = std::fmaf(dz, dz, std::fmaf(dy, dy, dx * dx));
                    if (d2 < sigma2) overlap = true;
                    if (d2 < well2) ++n_well;
                }
                w[t] = overlap ? 0 : Q[n_well < 31 ? n_well : 31];
                if (!overlap) ++m;
                W += w[t];
            }
            ++n_steps;
            if (mrow) mrow[s - 1] = (uint8_t)m;
            if (m == 0) {
                alive = false; h = digest_fold(h, 0, 0xFF);
                for (int32_t q = s; q < N; ++q) r[3*q] = r[3*q+1] = r[3*q+2] = 0.0f;
                break;
            }
            lnW += std::log((double)W * 0x1p-16);
            const uint64_t target = scaled_target(selection_word(seed, chain, (uint32_t)s), W);
            int32_t t = 0;
            uint64_t cum = w[0];
            while (cum <= target) cum += w[++t];
            r[3*s] = trial[3*t]; r[3*s+1] = trial[3*t+1]; r[3*s+2] = trial[3*t+2];
            h = digest_fold(h, (uint32_t)m, (uint32_t)t);
        }

        double ree2 = 0.0, rg2 = 0.0;
        if (alive) {
            double cx = 0.0, cy = 0.0, cz = 0.0;
            for (int32_t q = 0; q < N; ++q) { cx += (double)r[3*q]; cy += (double)r[3*q+1]; cz += (double)r[3*q+2]; }
            cx /= (double)N; cy /= (double)N; cz /= (double)N;
            double acc = 0.0;
            for (int32_t q = 0; q < N; ++q) {
                const double ax = (double)r[3*q] - cx, ay = (double)r[3*q+1] - cy, az = (double)r[3*q+2] - cz;
                acc += ax*ax + ay*ay + az*az;
            }
            rg2 = acc / (double)N;
            const double ex = (double)r[3*(N-1)], ey = (double)r[3*(N-1)+1], ez = (double)r[3*(N-1)+2];
            ree2 = ex*ex + ey*ey + ez*ez;
        } else {
            lnW = -std::numeric_limits<double>::infinity();
        }
        res.push_back(ChainResult{lnW, ree2, rg2, alive});
        dxor ^= h; dsum += h;
        if (out) {
            if (out->lnW) out->lnW[i] = lnW;
            if (out->alive) out->alive[i] = alive ? 1 : 0;
            if (out->digest) out->digest[i] = h;
            if (out->ree2) out->ree2[i] = ree2;
            if (out->rg2) out->rg2[i] = rg2;
            if (out->conf) std::memcpy((float*)out->conf + i * (size_t)N * 3, r.data(), (size_t)N * 3 * sizeof(float));
        }
    }
    ensemble(summary, res, true, 0.0, n_steps, dxor, dsum);
    return 0;
}

// ---------------------------------------------------------------------------------------------
// PERM, the pruned-enriched Rosenbluth method. The paper names it only as the topic of its
// supplement ("Parallel implementation of PERM on GPU"), which is not available: what follows is the
// published algorithm (P. Grassberger, Phys. Rev. E 56, 3682 (1997)) in its depth-first recursive form, with the
// population-control thresholds GIVEN by the caller (readings A22-A24) so that a tour is a pure function
// of (seed, tour id, thresholds):
//   step(n, lnW): the chain has n monomers and weight W. If n = N it is a leaf: the tour's sums take W, W Ree2, W Rg2.
//     Otherwise node = next node number of the tour; m = free neighbours (Alg. 1); m = 0: dead end, return.
//     W' = W m; the monomer goes to the ((u m) >> 32)-th free site, u = selection word (seed, tour, node + 1) of 3.1.
//     Population control at the new length n + 1 < N:  lnW' > ln_hi[n+1]: enrichment, two copies of weight W'/2 each;
//     lnW' < ln_lo[n+1]: pruning, killed if the coin word (Philox counter (tour, node >> 2, 2), word node & 3) is < 2^31,
//     else the weight doubles. Then step(n + 1, .) once per copy. A tour that reaches max_nodes nodes stops (flag 2).
// With ln_lo = -inf, ln_hi = +inf a tour IS the Rosenbluth chain of the same id (same words, same decisions).
// The estimate of Z_N is the mean over tours of S = sum of leaf weights; E[S] = c_{N-1} for any thresholds.
// ---------------------------------------------------------------------------------------------
struct PermTour {
    int32_t N; uint64_t seed, tour; const double* ln_lo; const double* ln_hi; double ln_ref; uint64_t max_nodes;
    std::vector<int32_t> r;
    uint64_t node = 0, leaves = 0, h = 0;
    bool capped = false;
    double S = 0.0, SR = 0.0, SG = 0.0;       // sums of exp(lnW - ln_ref) (x Ree2, x Rg2) over the leaves, depth-first order

    void step(int32_t n, double lnW) {
        if (capped) return;
        if (n == N) {
            int64_t sx = 0, sy = 0, sz = 0, s2 = 0;
            for (int32_t q = 0; q < N; ++q) {
                const int64_t x = r[3*q], y = r[3*q+1], z = r[3*q+2];
                sx += x; sy += y; sz += z; s2 += x*x + y*y + z*z;
            }
            const int64_t ex = r[3*(N-1)], ey = r[3*(N-1)+1], ez = r[3*(N-1)+2];
            const double ree2 = (double)(ex*ex + ey*ey + ez*ez);
            const double rg2 = (double)((int64_t)N * s2 - (sx*sx + sy*sy + sz*sz)) / ((double)N * (double)N);
            const double w = std::exp(lnW - ln_ref);
            S += w; SR += w * ree2; SG += w * rg2; ++leaves;
            return;
        }
        if (node >= max_nodes) { capped = true; return; }
        const uint64_t id = node++;
        int32_t free_dirs[6];
        const int32_t m = oracle_lattice_free_dirs(r.data(), n, free_dirs);
        if (m == 0) { h = digest_fold(h, 0, 0xFF); return; }
        lnW += std::log((double)m);
        const uint32_t u = selection_word(seed, tour, (uint32_t)(id + 1));
        const int32_t d = free_dirs[(uint32_t)(((uint64_t)u * (uint64_t)m) >> 32)];
        for (int a = 0; a < 3; ++a) r[3*n+a] = r[3*(n-1)+a] + E[d][a];
        int copies = 1;
        uint32_t event = 0;
        if (n + 1 < N) {
            if (lnW > ln_hi[n + 1]) { copies = 2; lnW -= std::log(2.0); event = 1; }
            else if (lnW < ln_lo[n + 1]) {
                const uint32_t ctr[4] = { (uint32_t)tour, (uint32_t)(tour >> 32), (uint32_t)(id >> 2), 2u };
                const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
                uint32_t w4[4];
                oracle_philox4x32_10(ctr, key, w4);
                if (w4[id & 3u] < 0x80000000u) { copies = 0; event = 3; } else { lnW += std::log(2.0); event = 2; }
            }
        }
        h = digest_fold(h, (uint32_t)m | (event << 4), (uint32_t)d);
        for (int c = 0; c < copies; ++c) {
            // the copy made at this length continues from r[0..n]; deeper levels only overwrote monomers > n
            for (int a = 0; a < 3; ++a) r[3*n+a] = r[3*(n-1)+a] + E[d][a];
            step(n + 1, lnW);
        }
    }
};

// Per-tour results use the per-chain fields: lnW = ln S (ln of the tour's summed leaf weights, -inf without a leaf),
// ree2 / rg2 = the tour's weighted means SR/S, SG/S, alive = 1 (some leaf), 0 (none), 2 (stopped at max_nodes).
// Summary: n_chains = tours, n_dead = tours without a leaf, n_steps_attempted = nodes, sums over tours of
// exp(lnS - L) (x ree2, x rg2, squared), L = largest lnS; mean_* = W-weighted means over all leaves, ln_mean_W = ln Z_N estimate.
int oracle_lattice_perm(int32_t N, uint64_t n_tours, uint64_t seed, uint64_t tour_offset, const double* ln_lo, const double* ln_hi,
                        double ln_ref, uint64_t max_nodes, const oracle_outputs* out, oracle_summary* summary)
{
    if (N < 2 || N > 4096 || n_tours == 0 || !ln_lo || !ln_hi || max_nodes == 0 || !std::isfinite(ln_ref)) return -1;
    std::vector<ChainResult> res;
    res.reserve(n_tours);
    uint64_t n_nodes = 0, dxor = 0, dsum = 0;
    for (uint64_t i = 0; i < n_tours; ++i) {
        PermTour t;
        t.N = N; t.seed = seed; t.tour = tour_offset + i; t.ln_lo = ln_lo; t.ln_hi = ln_hi; t.ln_ref = ln_ref; t.max_nodes = max_nodes;
        t.r.assign((size_t)N * 3, 0);
        t.h = digest_init();
        t.step(1, 0.0);
        const bool have = t.S > 0.0;
        const double lnS = have ? ln_ref + std::log(t.S) : -std::numeric_limits<double>::infinity();
        const double ree2 = have ? t.SR / t.S : 0.0, rg2 = have ? t.SG / t.S : 0.0;
        res.push_back(ChainResult{lnS, ree2, rg2, have});
        n_nodes += t.node; dxor ^= t.h; dsum += t.h;
        if (out) {
            if (out->lnW) out->lnW[i] = lnS;
            if (out->alive) out->alive[i] = t.capped ? 2 : (have ? 1 : 0);
            if (out->digest) out->digest[i] = t.h;
            if (out->ree2) out->ree2[i] = ree2;
            if (out->rg2) out->rg2[i] = rg2;
        }
    }
    ensemble(summary, res, true, 0.0, n_nodes, dxor, dsum);
    return 0;
}

}  // extern "C"
