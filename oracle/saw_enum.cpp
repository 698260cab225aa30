// saw_enum.cpp -- TEST INFRASTRUCTURE. Brute-force enumeration of all n-step self-avoiding walks
// on the simple cubic lattice (depth-first, own occupancy grid), used to pin the lattice oracle:
//
//   * c_n = number of n-step SAWs (known series, tests/golden/saw_cubic_counts.txt)
//   * exact uniform-SAW means <Ree2> = sum_w Ree2 / c_n and <Rg2> = sum_w N^2 Rg2 / (N^2 c_n),
//     the values the W-weighted Rosenbluth averages (Eq. 2) must converge to
//   * the exact survival identity  sum_{w in SAW_n} 1/W(w) = P_alive(n)  (Eq. 3, PAPER.md:58-60:
//     "this walk is generated with probability P_n = 1/W_n"), with W(w) = prod_s m_s(w) computed
//     by the ORACLE's free-site routine (oracle_lattice_free_dirs in rosen_oracle.cpp), i.e. a
//     non-statistical test of that routine over every walk. W is always 2^a 3^b 5^c, so the
//     caller gets an exact histogram over (a,b,c) and sums it in rational arithmetic.
//
// The enumerator decides self-avoidance with its own grid, never with the oracle's scan.

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

extern "C" int32_t oracle_lattice_free_dirs(const int32_t* r, int32_t s, int32_t free_dirs[6]);
extern "C" int32_t oracle_lattice_model_step(const int32_t* r, int32_t s, int32_t z, const uint64_t Q[32], uint64_t w[26]);
extern "C" void oracle_model_table(double beta_eps, uint64_t Q[32]);

namespace {

struct Enum {
    int n;                      // steps
    int side;                   // grid side 2n+1
    std::vector<uint8_t> occ;   // own occupancy grid
    std::vector<int32_t> r;     // walk so far [n+1][3]
    int ea[64], eb[64], ec[64]; // cumulative exponents of 2,3,5 in W along the path
    uint64_t count = 0, sum_ree2 = 0, sum_n2rg2 = 0;
    uint64_t* hist;             // [(2n+1)][(n+1)][(n+1)] counts by (a,b,c)
    int fix_first;

    size_t cell(int x, int y, int z) const { return ((size_t)(x + n) * side + (size_t)(y + n)) * side + (size_t)(z + n); }

    void leaf() {
        const int N = n + 1;
        int64_t sx = 0, sy = 0, sz = 0, s2 = 0;
        for (int q = 0; q < N; ++q) {
            const int64_t x = r[3*q], y = r[3*q+1], z = r[3*q+2];
            sx += x; sy += y; sz += z; s2 += x*x + y*y + z*z;
        }
        const int64_t x = r[3*n], y = r[3*n+1], z = r[3*n+2];
        ++count;
        sum_ree2 += (uint64_t)(x*x + y*y + z*z);
        sum_n2rg2 += (uint64_t)((int64_t)N * s2 - (sx*sx + sy*sy + sz*sz));
        hist[((size_t)ea[n] * (n + 1) + eb[n]) * (n + 1) + ec[n]] += 1;
    }

    // s monomers placed (indices 0..s-1); place monomer s.
    void grow(int s) {
        if (s == n + 1) { leaf(); return; }
        int32_t fd[6];
        const int m = oracle_lattice_free_dirs(r.data(), s, fd);   // the routine under test
        if (m == 0) return;                                        // trapped: contributes to no n-step SAW
        static const int f2[7] = {0, 0, 1, 0, 2, 0, 1}, f3[7] = {0, 0, 0, 1, 0, 0, 1}, f5[7] = {0, 0, 0, 0, 0, 1, 0};
        ea[s] = ea[s-1] + f2[m]; eb[s] = eb[s-1] + f3[m]; ec[s] = ec[s-1] + f5[m];
        static const int E[6][3] = { {1,0,0}, {-1,0,0}, {0,1,0}, {0,-1,0}, {0,0,1}, {0,0,-1} };
        int extended = 0;
        for (int d = 0; d < 6; ++d) {
            if (s == 1 && fix_first && d != 0) continue;
            const int x = r[3*(s-1)] + E[d][0], y = r[3*(s-1)+1] + E[d][1], z = r[3*(s-1)+2] + E[d][2];
            const size_t c = cell(x, y, z);
            if (occ[c]) continue;                                  // own self-avoidance test
            ++extended;
            occ[c] = 1; r[3*s] = x; r[3*s+1] = y; r[3*s+2] = z;
            grow(s + 1);
            occ[c] = 0;
        }
        if (!(s == 1 && fix_first) && extended != m) inconsistent = true;   // grid and oracle scan must agree
    }
    bool inconsistent = false;
};

}  // namespace

extern "C" {

// Enumerate all n-step SAWs (1 <= n <= 16). If fix_first != 0 only walks whose first step is +x
// are visited (multiply every returned count by 6). hist must hold (2n+1)(n+1)(n+1) zeroed
// uint64. Returns 0, -1 on bad arguments, -2 if the oracle's free-site count ever disagreed
// with the enumerator's own grid.
int oracle_saw_enumerate(int32_t n, int32_t fix_first, uint64_t* count, uint64_t* sum_ree2,
                         uint64_t* sum_n2rg2, uint64_t* hist)
{
    if (n < 1 || n > 16 || !hist) return -1;
    Enum e;
    e.n = n; e.side = 2 * n + 1; e.fix_first = fix_first; e.hist = hist;
    e.occ.assign((size_t)e.side * e.side * e.side, 0);
    e.r.assign((size_t)(n + 1) * 3, 0);
    e.ea[0] = e.eb[0] = e.ec[0] = 0;
    e.occ[e.cell(0, 0, 0)] = 1;
    e.grow(1);
    if (count) *count = e.count;
    if (sum_ree2) *sum_ree2 = e.sum_ree2;
    if (sum_n2rg2) *sum_n2rg2 = e.sum_n2rg2;
    return e.inconsistent ? -2 : 0;
}

}  // extern "C"

// Model enumerator (z = 6 or 26 trial set, contact energy): depth-first over all n-step SAWs with its OWN
// occupancy grid, own direction table and own contact count (pairs |i - j| > 1 on neighbouring sites, counted from the
// definition over the whole walk). For every walk w it accumulates
//   count              1
//   sum_boltz          q^contacts(w)                      (q = exp(beta_eps) in fp64: the exact partition sum Z_n)
//   sum_boltz_ree2     q^contacts(w) Ree2(w)
//   sum_quant          prod_s Q[c_s(w)] 2^-16              (what E[W] of the fixed-point Rosenbluth scheme converges to)
//   sum_prob           prod_s w_s[d_s] / W_s               (probability that the ORACLE's step routine grows w;
//                                                           summed over all walks = P_alive(n): non-statistical pin)
// with c_s = contacts the monomer placed at step s makes; the last two use oracle_lattice_model_step (routine under test).
namespace {
struct EnumM {
    int n, z, side;
    std::vector<uint8_t> occ;
    std::vector<int32_t> r;
    uint64_t Q[32];
    double q;
    double count = 0, sum_boltz = 0, sum_boltz_ree2 = 0, sum_quant = 0, sum_prob = 0;
    bool inconsistent = false;
    int dirs[26][3];
    size_t cell(int x, int y, int zc) const { return ((size_t)(x + n) * side + (size_t)(y + n)) * side + (size_t)(zc + n); }
    bool adjacent(int i, int j) const {
        const int dx = std::abs(r[3*i] - r[3*j]), dy = std::abs(r[3*i+1] - r[3*j+1]), dz = std::abs(r[3*i+2] - r[3*j+2]);
        return z == 6 ? dx + dy + dz == 1 : (dx <= 1 && dy <= 1 && dz <= 1);
    }
    void grow(int s, double quant, double prob) {
        if (s == n + 1) {
            int contacts = 0;
            for (int i = 0; i <= n; ++i) for (int j = i + 2; j <= n; ++j) if (adjacent(i, j)) ++contacts;
            const double bw = std::pow(q, contacts);
            const double x = r[3*n], y = r[3*n+1], zz = r[3*n+2];
            count += 1; sum_boltz += bw; sum_boltz_ree2 += bw * (x*x + y*y + zz*zz); sum_quant += quant; sum_prob += prob;
            return;
        }
        uint64_t w[26];
        const int m = oracle_lattice_model_step(r.data(), s, z, Q, w);
        uint64_t W = 0;
        for (int d = 0; d < z; ++d) W += w[d];
        int extended = 0;
        for (int d = 0; d < z; ++d) {
            const int x = r[3*(s-1)] + dirs[d][0], y = r[3*(s-1)+1] + dirs[d][1], zc = r[3*(s-1)+2] + dirs[d][2];
            const size_t c = cell(x, y, zc);
            if (occ[c]) { if (w[d] != 0) inconsistent = true; continue; }
            if (w[d] == 0) { inconsistent = true; continue; }
            ++extended;
            occ[c] = 1; r[3*s] = x; r[3*s+1] = y; r[3*s+2] = zc;
            grow(s + 1, quant * ((double)w[d] * 0x1p-16), prob * ((double)w[d] / (double)W));
            occ[c] = 0;
        }
        if (extended != m) inconsistent = true;
    }
};
}  // namespace

extern "C" int oracle_saw_enumerate_model(int32_t n, int32_t z, double beta_eps, double out[5])
{
    if (n < 1 || n > 12 || (z != 6 && z != 26) || !out) return -1;
    EnumM e;
    e.n = n; e.z = z; e.side = 2 * n + 1; e.q = std::exp(beta_eps);
    oracle_model_table(beta_eps, e.Q);
    // own direction table, written out independently of the oracle's model_dir
    int nd = 0;
    if (z == 6) {
        const int E6[6][3] = { {1,0,0}, {-1,0,0}, {0,1,0}, {0,-1,0}, {0,0,1}, {0,0,-1} };
        for (; nd < 6; ++nd) for (int a = 0; a < 3; ++a) e.dirs[nd][a] = E6[nd][a];
    } else {
        for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
            if (dx == 0 && dy == 0 && dz == 0) continue;
            e.dirs[nd][0] = dx; e.dirs[nd][1] = dy; e.dirs[nd][2] = dz; ++nd;
        }
    }
    e.occ.assign((size_t)e.side * e.side * e.side, 0);
    e.r.assign((size_t)(n + 1) * 3, 0);
    e.occ[e.cell(0, 0, 0)] = 1;
    e.grow(1, 1.0, 1.0);
    out[0] = e.count; out[1] = e.sum_boltz; out[2] = e.sum_boltz_ree2; out[3] = e.sum_quant; out[4] = e.sum_prob;
    return e.inconsistent ? -2 : 0;
}
