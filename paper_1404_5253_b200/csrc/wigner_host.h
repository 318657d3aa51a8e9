// wigner_host.h -- host-side angular-momentum algebra for wpcd_channels_create.
//
// Part of the PRODUCT path (libwpcd); shares nothing with oracle/.  Computes the
// coefficients g^{l1 l1' k}_{gamma gamma'} of (A4) (step 1 of the
// scheme, PAPER.md:310 -- "negligible" host work) in the reading R1/R2 of DESIGN.md.
// Racah single-sum formulae evaluated in long double with a factorial table;
// all momenta DOUBLED (two_j) so half-integers are ints.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <algorithm>
#include <array>
#include <map>
#include <vector>

namespace wpcd_host {

struct Factorials {
    long double f[96];
    Factorials() { f[0] = 1.0L; for (int i = 1; i < 96; ++i) f[i] = f[i - 1] * (long double)i; }
    long double operator()(int n) const { return f[n]; }
};
inline const Factorials& fact() { static Factorials F; return F; }

inline bool triangle(int a2, int b2, int c2) {
    return ((a2 + b2 + c2) & 1) == 0 && c2 >= std::abs(a2 - b2) && c2 <= a2 + b2;
}

inline long double delta_sq(int a2, int b2, int c2) {
    const Factorials& F = fact();
    return F((a2 + b2 - c2) / 2) * F((a2 - b2 + c2) / 2) * F((-a2 + b2 + c2) / 2) / F((a2 + b2 + c2) / 2 + 1);
}

// {j1 j2 j3; j4 j5 j6}
inline long double six_j(int j1, int j2, int j3, int j4, int j5, int j6) {
    if (!(triangle(j1, j2, j3) && triangle(j1, j5, j6) && triangle(j4, j2, j6) && triangle(j4, j5, j3))) return 0.0L;
    const Factorials& F = fact();
    int a1 = (j1 + j2 + j3) / 2, a2 = (j1 + j5 + j6) / 2, a3 = (j4 + j2 + j6) / 2, a4 = (j4 + j5 + j3) / 2;
    int b1 = (j1 + j2 + j4 + j5) / 2, b2 = (j2 + j3 + j5 + j6) / 2, b3 = (j3 + j1 + j6 + j4) / 2;
    int lo = a1; if (a2 > lo) lo = a2; if (a3 > lo) lo = a3; if (a4 > lo) lo = a4;
    int hi = b1; if (b2 < hi) hi = b2; if (b3 < hi) hi = b3;
    long double sum = 0.0L;
    for (int t = lo; t <= hi; ++t) {
        long double term = F(t + 1) / (F(t - a1) * F(t - a2) * F(t - a3) * F(t - a4) * F(b1 - t) * F(b2 - t) * F(b3 - t));
        sum += (t & 1) ? -term : term;
    }
    return sum * sqrtl(delta_sq(j1, j2, j3) * delta_sq(j1, j5, j6) * delta_sq(j4, j2, j6) * delta_sq(j4, j5, j3));
}

// {j1 j2 j3; j4 j5 j6; j7 j8 j9} by the single sum over 6j triple products
inline long double nine_j(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9) {
    if (!(triangle(j1, j2, j3) && triangle(j4, j5, j6) && triangle(j7, j8, j9) &&
          triangle(j1, j4, j7) && triangle(j2, j5, j8) && triangle(j3, j6, j9))) return 0.0L;
    int lo = std::abs(j1 - j9); if (std::abs(j4 - j8) > lo) lo = std::abs(j4 - j8); if (std::abs(j2 - j6) > lo) lo = std::abs(j2 - j6);
    int hi = j1 + j9; if (j4 + j8 < hi) hi = j4 + j8; if (j2 + j6 < hi) hi = j2 + j6;
    long double sum = 0.0L;
    for (int x = lo; x <= hi; x += 2) {
        long double term = (long double)(x + 1) * six_j(j1, j4, j7, j8, j9, x) * six_j(j2, j5, j8, j4, x, j6) * six_j(j3, j6, j9, x, j1, j2);
        sum += (x & 1) ? -term : term;
    }
    return sum;
}

// <a 0 b 0 | c 0>, integer a, b, c
inline long double cg000(int a, int b, int c) {
    if (((a + b + c) & 1) || c < std::abs(a - b) || c > a + b) return 0.0L;
    const Factorials& F = fact();
    int g = (a + b + c) / 2;
    long double tj = sqrtl(F(2 * g - 2 * a) * F(2 * g - 2 * b) * F(2 * g - 2 * c) / F(2 * g + 1)) * F(g) / (F(g - a) * F(g - b) * F(g - c));
    if (g & 1) tj = -tj;
    long double v = sqrtl((long double)(2 * c + 1)) * tj;
    return ((a - b) & 1) ? -v : v;
}

struct Channel { int l, s, j, t, lam, two_I; };

// eq. (5) with l+s+t odd, j <= j_max, (-1)^{l+lam} = parity; order documented in wpcd.h
inline std::vector<Channel> enumerate_channels(int two_J, int parity, int j_max) {
    std::vector<Channel> out;
    for (int j = 0; j <= j_max; ++j)
        for (int s = 0; s <= 1; ++s)
            for (int l = std::abs(j - s); l <= j + s; ++l) {
                int t = 1 - ((l + s) & 1);
                for (int two_I = std::abs(two_J - 2 * j); two_I <= two_J + 2 * j; two_I += 2)
                    for (int lam = (two_I - 1) / 2; lam <= (two_I + 1) / 2; ++lam) {
                        if (lam < 0) continue;
                        if ((((l + lam) & 1) ? -1 : 1) != parity) continue;
                        out.push_back({l, s, j, t, lam, two_I});
                    }
            }
    return out;
}

// orbital part of (A4) for one L
inline long double orbital(int l, int lam, int lp, int lamp, int L, int l1, int l1p, int k) {
    const Factorials& F = fact();
    int l2 = l - l1, l2p = lp - l1p;
    long double ff = 0.0L;
    for (int f = std::abs(l1 - lam); f <= l1 + lam; ++f) {
        long double c1 = cg000(l1, lam, f); if (c1 == 0.0L) continue;
        long double c2 = cg000(k, l1p, f); if (c2 == 0.0L) continue;
        long double s1 = six_j(2 * l2, 2 * l1, 2 * l, 2 * lam, 2 * L, 2 * f); if (s1 == 0.0L) continue;
        for (int fp = std::abs(l2p - lamp); fp <= l2p + lamp; ++fp) {
            long double c3 = cg000(l2p, lamp, fp); if (c3 == 0.0L) continue;
            long double c4 = cg000(k, l2, fp); if (c4 == 0.0L) continue;
            ff += six_j(2 * l1p, 2 * l2p, 2 * lp, 2 * lamp, 2 * L, 2 * fp) * s1 * c3 * c1 *
                  six_j(2 * fp, 2 * l1p, 2 * L, 2 * f, 2 * l2, 2 * k) * c2 * c4;
        }
    }
    long double geom = (long double)(2 * k + 1) * powl(0.5L, l2p + l1) *
                       sqrtl(F(2 * l + 1) / (F(2 * l1) * F(2 * l2))) * sqrtl(F(2 * lp + 1) / (F(2 * l1p) * F(2 * l2p)));
    return geom * ff;
}

struct Term { int k, l1, l1p; double g; };
struct Pair { int gamma, gammap; std::vector<Term> terms; };

// All coupled pairs with their nonzero terms (|g| > 1e-14), sorted by (gamma, gamma').
inline std::vector<Pair> g_table(const std::vector<Channel>& ch, int two_J, int two_T) {
    std::vector<Pair> pairs;
    auto hat = [](int x) { return (long double)(2 * x + 1); };
    // The orbital part depends on (l, lambda, l', lambda'; L, l1, l1', k) only -- not on the spins, j, I of the channels -- so
    // it is tabulated once per distinct (l, lambda, l', lambda') and reused by every channel pair that carries these labels
    // (62 channels share ~20 distinct (l, lambda) for the nd tables of j <= 3: a tenth of the evaluations).
    struct OrbitalBlock { int Llo, Lhi, K; std::vector<long double> v; };      // v[((L - Llo) (l+1) + l1) (l'+1) + l1'] K + k]
    std::map<std::array<int, 4>, OrbitalBlock> blocks;
    auto block_of = [&](int l, int lam, int lp, int lamp) -> const OrbitalBlock& {
        const std::array<int, 4> key = {l, lam, lp, lamp};
        auto it = blocks.find(key);
        if (it != blocks.end()) return it->second;
        OrbitalBlock blk;
        blk.Llo = std::max(std::abs(l - lam), std::abs(lp - lamp));
        blk.Lhi = std::min(l + lam, lp + lamp);
        blk.K = l + lam + lp + lamp + 1;                               // k <= min(l1 + lambda + l1', l2' + lambda' + l2) < K
        const int nL = blk.Lhi >= blk.Llo ? blk.Lhi - blk.Llo + 1 : 0;
        blk.v.assign((size_t)nL * (l + 1) * (lp + 1) * blk.K, 0.0L);
        for (int L = blk.Llo; L <= blk.Lhi; ++L)
            for (int l1 = 0; l1 <= l; ++l1)
                for (int l1p = 0; l1p <= lp; ++l1p) {
                    const int l2 = l - l1, l2p = lp - l1p;
                    const int kmax = std::min(l1 + lam + l1p, l2p + lamp + l2);
                    for (int k = 0; k <= kmax; ++k)
                        blk.v[((size_t)((L - blk.Llo) * (l + 1) + l1) * (lp + 1) + l1p) * blk.K + k] = orbital(l, lam, lp, lamp, L, l1, l1p, k);
                }
        return blocks.emplace(key, std::move(blk)).first->second;
    };
    // the 9j symbol of a channel for every (L, S) it can take part in: {l s j; lambda 1/2 I; L S J}
    int Lmax = 0;
    for (const Channel& c : ch) Lmax = std::max(Lmax, c.l + c.lam);
    std::vector<long double> nj(ch.size() * (size_t)(Lmax + 1) * 2, 0.0L);
    for (size_t a = 0; a < ch.size(); ++a)
        for (int L = std::abs(ch[a].l - ch[a].lam); L <= ch[a].l + ch[a].lam; ++L)
            for (int si = 0; si < 2; ++si)
                nj[(a * (Lmax + 1) + L) * 2 + si] = nine_j(2 * ch[a].l, 2 * ch[a].s, 2 * ch[a].j, 2 * ch[a].lam, 1, ch[a].two_I, 2 * L, 1 + 2 * si, two_J);
    for (size_t a = 0; a < ch.size(); ++a)
        for (size_t b = 0; b < ch.size(); ++b) {
            const Channel &c = ch[a], &d = ch[b];
            long double iso = six_j(1, 1, 2 * c.t, 1, two_T, 2 * d.t);
            if (iso == 0.0L) continue;
            long double pref = -sqrtl(hat(c.l) * hat(c.s) * hat(c.j) * hat(c.t) * hat(c.lam) * (c.two_I + 1) *
                                      hat(d.l) * hat(d.s) * hat(d.j) * hat(d.t) * hat(d.lam) * (d.two_I + 1));
            // spin/9j weights per (L,S)
            int Llo = std::abs(c.l - c.lam); if (std::abs(d.l - d.lam) > Llo) Llo = std::abs(d.l - d.lam);
            int Lhi = c.l + c.lam; if (d.l + d.lam < Lhi) Lhi = d.l + d.lam;
            std::vector<long double> wL(Lhi >= Llo ? Lhi - Llo + 1 : 0, 0.0L);
            bool any = false;
            for (int L = Llo; L <= Lhi; ++L)
                for (int two_S = 1; two_S <= 3; two_S += 2) {
                    long double spin = six_j(1, 1, 2 * c.s, 1, two_S, 2 * d.s);
                    if (spin == 0.0L) continue;
                    long double n1 = nj[(a * (Lmax + 1) + L) * 2 + (two_S >> 1)];
                    if (n1 == 0.0L) continue;
                    long double n2 = nj[(b * (Lmax + 1) + L) * 2 + (two_S >> 1)];
                    wL[L - Llo] += (long double)(2 * L + 1) * (two_S + 1) * spin * n1 * n2;
                    any = any || (n2 != 0.0L);
                }
            if (!any) continue;
            Pair pr{(int)a, (int)b, {}};
            const OrbitalBlock& blk = block_of(c.l, c.lam, d.l, d.lam);
            for (int l1 = 0; l1 <= c.l; ++l1)
                for (int l1p = 0; l1p <= d.l; ++l1p) {
                    int l2 = c.l - l1, l2p = d.l - l1p;
                    int kmax = l1 + c.lam + l1p; if (l2p + d.lam + l2 < kmax) kmax = l2p + d.lam + l2;
                    for (int k = 0; k <= kmax; ++k) {
                        long double tot = 0.0L;
                        for (int L = Llo; L <= Lhi; ++L)
                            if (wL[L - Llo] != 0.0L)
                                tot += wL[L - Llo] * blk.v[((size_t)((L - blk.Llo) * (c.l + 1) + l1) * (d.l + 1) + l1p) * blk.K + k];
                        double g = (double)(pref * iso * tot);
                        if (std::fabs(g) > 1e-14) pr.terms.push_back({k, l1, l1p, g});
                    }
                }
            if (!pr.terms.empty()) pairs.push_back(std::move(pr));
        }
    return pairs;
}

// n-point Gauss-Legendre nodes/weights on [-1,1] by Newton iteration on P_n (ascending nodes)
inline void gauss_legendre(int n, double* xi, double* w) {
    for (int i = 0; i < n; ++i) {
        long double x = cosl(3.14159265358979323846264338327950288L * (i + 0.75L) / (n + 0.5L));
        long double dp = 1.0L;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1.0L, p1 = x;
            for (int k = 2; k <= n; ++k) { long double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
            if (n == 1) { p0 = 1.0L; p1 = x; }
            dp = n * (x * p1 - p0) / (x * x - 1.0L);
            long double dx = p1 / dp;
            x -= dx;
            if (fabsl(dx) < 1e-19L) break;
        }
        {   // derivative at the converged node
            long double p0 = 1.0L, p1 = x;
            for (int k = 2; k <= n; ++k) { long double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
            dp = n * (x * p1 - p0) / (x * x - 1.0L);
        }
        xi[n - 1 - i] = (double)x;
        w[n - 1 - i] = (double)(2.0L / ((1.0L - x * x) * dp * dp));
    }
}

}  // namespace wpcd_host
