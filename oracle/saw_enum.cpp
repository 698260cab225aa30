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

#include <cstdint>
#include <cstring>
#include <vector>

extern "C" int32_t oracle_lattice_free_dirs(const int32_t* r, int32_t s, int32_t free_dirs[6]);

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
