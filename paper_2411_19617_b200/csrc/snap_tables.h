// snap_tables.h -- host-side table construction for the CUDA bispectrum path.
//
// Everything here is plain host C++: the list of (j1,j2,j) triples (Eq. (26), PAPER.md:263 fixes its length),
// the half-column storage map of U_tot, the binomial normalisation of the polynomial form of the Wigner-U
// recursion, the Clebsch-Gordan table, and the cost-sorted work order of the Z contraction.
// It shares no code with oracle/ (the oracle has its own CG and its own enumeration).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

namespace mala {

// ---- compile-time helpers shared by host tables and the specialised kernels -------------------------------
// half-column storage: level J keeps columns mb = 0..J/2, each with J+1 rows; element (J, mb, ma) lives at
// uhalf_off(J) + mb*(J+1) + ma.  The other columns follow from u[J-ma][J-mb] = (-1)^(ma-mb) conj(u[ma][mb]).
constexpr int uhalf_off(int J) {
    int o = 0;
    for (int K = 0; K < J; K++) o += (K + 1) * (K / 2 + 1);
    return o;
}
constexpr int uhalf_size(int twojmax) { return uhalf_off(twojmax + 1); }

struct Triple {
    int j1, j2, j;
};

constexpr int triple_count(int twojmax) {
    int n = 0;
    for (int j1 = 0; j1 <= twojmax; j1++)
        for (int j2 = 0; j2 <= j1; j2++)
            for (int j = j1 - j2; j <= (twojmax < j1 + j2 ? twojmax : j1 + j2); j += 2)
                if (j >= j1) n++;
    return n;
}

// idx-th triple in output order (reading #7: j1 outer, j2, j inner, j >= j1 >= j2)
constexpr Triple triple_at(int twojmax, int idx) {
    int n = 0;
    for (int j1 = 0; j1 <= twojmax; j1++)
        for (int j2 = 0; j2 <= j1; j2++)
            for (int j = j1 - j2; j <= (twojmax < j1 + j2 ? twojmax : j1 + j2); j += 2)
                if (j >= j1) {
                    if (n == idx) return Triple{j1, j2, j};
                    n++;
                }
    return Triple{-1, -1, -1};
}

// offset of triple idx in the dense CG table: per triple a (J2+1) x (J1+1) block, entry [m2][m1]
constexpr int cg_block_off(int twojmax, int idx) {
    int o = 0;
    for (int i = 0; i < idx; i++) {
        Triple t = triple_at(twojmax, i);
        o += (t.j1 + 1) * (t.j2 + 1);
    }
    return o;
}

// ---- Clebsch-Gordan coefficient (doubled arguments), Condon-Shortley phases ---------------------------------
// Racah's single-sum closed form evaluated in long double with a factorial table; every factorial that occurs
// for twojmax <= 16 is below 34! and the sum has at most 17 terms, so the result is correct to ~1 ulp of double.
inline long double lfactorial(int n) {
    static long double tab[64];
    static bool init = false;
    if (!init) {
        tab[0] = 1.0L;
        for (int i = 1; i < 64; i++) tab[i] = tab[i - 1] * (long double)i;
        init = true;
    }
    return tab[n];
}

inline double clebsch_gordan(int J1, int M1, int J2, int M2, int J, int M) {
    if (J1 < 0 || J2 < 0 || J < 0) return 0.0;
    if (M != M1 + M2) return 0.0;
    if (((J1 + J2 + J) & 1) != 0) return 0.0;
    if (J > J1 + J2 || J < std::abs(J1 - J2)) return 0.0;
    if (std::abs(M1) > J1 || std::abs(M2) > J2 || std::abs(M) > J) return 0.0;
    if (((J1 + M1) & 1) || ((J2 + M2) & 1) || ((J + M) & 1)) return 0.0;
    // half-integer bookkeeping in plain integers
    const int s_abc = (J1 + J2 + J) / 2;      // j1 + j2 + j
    const int p1 = (J1 + M1) / 2, q1 = (J1 - M1) / 2;
    const int p2 = (J2 + M2) / 2, q2 = (J2 - M2) / 2;
    const int p = (J + M) / 2, q = (J - M) / 2;
    const int t12 = s_abc - J;                // j1 + j2 - j
    const int t1 = s_abc - J2;                // j1 - j2 + j
    const int t2 = s_abc - J1;                // -j1 + j2 + j
    long double tri = lfactorial(t12) * lfactorial(t1) * lfactorial(t2) / lfactorial(s_abc + 1);
    long double mfac = lfactorial(p1) * lfactorial(q1) * lfactorial(p2) * lfactorial(q2) * lfactorial(p) * lfactorial(q);
    // sum over k with all six factorial arguments non-negative
    const int e1 = (J - J2 + M1) / 2;         // j - j2 + m1
    const int e2 = (J - J1 - M2) / 2;         // j - j1 - m2
    const int kmin = std::max(0, std::max(-e1, -e2));
    const int kmax = std::min(t12, std::min(q1, p2));
    long double sum = 0.0L;
    for (int k = kmin; k <= kmax; k++) {
        long double den = lfactorial(k) * lfactorial(t12 - k) * lfactorial(q1 - k) * lfactorial(p2 - k) *
                          lfactorial(e1 + k) * lfactorial(e2 + k);
        sum += ((k & 1) ? -1.0L : 1.0L) / den;
    }
    return (double)(sqrtl((long double)(J + 1) * tri * mfac) * sum);
}

// ---- runtime tables -----------------------------------------------------------------------------------------
struct SnapTables {
    int twojmax = 0;
    int ntriples = 0;
    int nelem = 0;                   // uhalf_size(twojmax)
    std::vector<int> triples;        // [ntriples*4]: j1, j2, j, cg offset
    std::vector<double> cg;          // dense blocks, [m2][m1] per triple; 0 where the resulting m is out of range
    std::vector<double> unorm;       // [nelem]: sqrt(C(J,mb)/C(J,ma)) -- polynomial form -> Wigner-U
    std::vector<int> udiag;          // [nelem]: 1 where ma == mb (self term)
    std::vector<int> order;          // [ntriples]: triple indices sorted by decreasing contraction cost
    std::vector<long long> cost;     // [ntriples]: product terms of the half-column contraction
    long long total_terms = 0;
};

inline double binom_d(int n, int k) {
    double r = 1.0;
    for (int i = 1; i <= k; i++) r = r * (double)(n - k + i) / (double)i;
    return std::floor(r + 0.5);
}

inline SnapTables build_tables(int twojmax) {
    SnapTables T;
    T.twojmax = twojmax;
    T.ntriples = triple_count(twojmax);
    T.nelem = uhalf_size(twojmax);
    int off = 0;
    for (int i = 0; i < T.ntriples; i++) {
        Triple t = triple_at(twojmax, i);
        T.triples.push_back(t.j1);
        T.triples.push_back(t.j2);
        T.triples.push_back(t.j);
        T.triples.push_back(off);
        const int sh = (t.j1 + t.j2 - t.j) / 2;
        for (int m2 = 0; m2 <= t.j2; m2++)
            for (int m1 = 0; m1 <= t.j1; m1++) {
                const int m = m1 + m2 - sh;
                double v = 0.0;
                if (m >= 0 && m <= t.j)
                    v = clebsch_gordan(t.j1, 2 * m1 - t.j1, t.j2, 2 * m2 - t.j2, t.j, 2 * m - t.j);
                T.cg.push_back(v);
            }
        off += (t.j1 + 1) * (t.j2 + 1);
        // cost model: product terms over half columns, middle column restricted to ma <= J/2
        long long terms = 0;
        for (int mb = 0; mb <= t.j / 2; mb++) {
            const bool mid = (t.j % 2 == 0) && (mb == t.j / 2);
            const int nb = std::min(t.j1, mb + sh) - std::max(0, mb + sh - t.j2) + 1;
            long long conv = 0;
            for (int m2 = 0; m2 <= t.j2; m2++)
                for (int m1 = 0; m1 <= t.j1; m1++) {
                    const int m = m1 + m2 - sh;
                    if (m >= 0 && m <= (mid ? t.j / 2 : t.j)) conv++;
                }
            terms += (long long)nb * conv;
        }
        T.cost.push_back(terms);
        T.total_terms += terms;
    }
    T.order.resize(T.ntriples);
    for (int i = 0; i < T.ntriples; i++) T.order[i] = i;
    std::stable_sort(T.order.begin(), T.order.end(), [&](int a, int b) { return T.cost[a] > T.cost[b]; });
    T.unorm.resize(T.nelem);
    T.udiag.resize(T.nelem);
    for (int J = 0; J <= twojmax; J++)
        for (int mb = 0; mb <= J / 2; mb++)
            for (int ma = 0; ma <= J; ma++) {
                const int e = uhalf_off(J) + mb * (J + 1) + ma;
                T.unorm[e] = std::sqrt(binom_d(J, mb) / binom_d(J, ma));
                T.udiag[e] = (ma == mb) ? 1 : 0;
            }
    return T;
}

}  // namespace mala
