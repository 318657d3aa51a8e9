/* perm_oracle.c -- CPU oracle for the permutation-operator matrix P0.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Plain FP64 C, written from
 * PAPER.md Appendix A; shares no code with the CUDA path.  Build:
 *   gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC perm_oracle.c -lm
 * (-ffp-contract=off: the overlap predicate is an IEEE +,-,*,/ contract, R6).
 *
 * Notation (A6/A7):
 *   row cell    (i ,j ): p  in [L2,U2] = [p_{i-1},p_i],    q  in [a,b] = [q_{j-1},q_j]
 *   column cell (i',j'): p' in [L1,U1] = [p_{i'-1},p_{i'}], q' in [c,d] = [q_{j'-1},q_{j'}]
 *   pi1 = sqrt(q^2 + q'^2/4 + q q' x) goes with p', pi2 = sqrt(q^2/4 + q'^2 + q q' x) with p (A2).
 *   In the (q,q') plane a point is written (s,t).
 *
 * Functions
 *   wpo_overlap        structural-nonzero predicate S (R6) + the polygon Pi
 *   wpo_geo_count/fill geometric CSR pattern (rows (i,j), columns (i',j') ascending)
 *   wpo_elements       values of listed geometric elements for all coupled channel
 *                      pairs by the rule R(n) (R7) applied to (A15)
 *   wpo_elements_rule  the same with the kink-split rule RS(n) (R14) when split == 1, with the rule RA(n)
 *                      (kink-split in phi and u, exact u-integral; s-wave term only; R15) when split == 2
 *   wpo_spmv           sequential CSR y = P0 x
 *
 * Pins: tests/test_oracle_*.py (Cartesian (A7) brute force, single-cell constant,
 * symmetric-state eigenvalue 2 g0, spectrum bound, symmetry, point sampling of
 * the theta-product for the pattern).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define WPO_MAXV 16 /* rectangle (4) + at most one new vertex per half-plane (6) */

typedef struct { double s, t; } wpo_pt;

/* The six half-planes of DESIGN.md R6; inside <=> value >= 0. */
static double halfplane(int m, double s, double t, double L1, double U1, double L2, double U2)
{
    switch (m) {
    case 0: return (s + 0.5 * t) - L1;   /* q + q'/2 >= L1   (pi1 can reach L1 from above) */
    case 1: return U1 - (s - 0.5 * t);   /* q - q'/2 <= U1 */
    case 2: return U1 - (0.5 * t - s);   /* q'/2 - q <= U1 */
    case 3: return (0.5 * s + t) - L2;   /* q/2 + q' >= L2 */
    case 4: return U2 - (t - 0.5 * s);   /* q' - q/2 <= U2 */
    default: return U2 - (0.5 * s - t);  /* q/2 - q' <= U2 */
    }
}

/* Sutherland-Hodgman clip of a convex polygon by half-plane m. */
static int clip_polygon(const wpo_pt* in, int n, wpo_pt* out, int m,
                        double L1, double U1, double L2, double U2)
{
    int no = 0;
    for (int e = 0; e < n; ++e) {
        wpo_pt P = in[e], Q = in[(e + 1) % n];
        double fP = halfplane(m, P.s, P.t, L1, U1, L2, U2);
        double fQ = halfplane(m, Q.s, Q.t, L1, U1, L2, U2);
        int inP = fP >= 0.0, inQ = fQ >= 0.0;
        if (inP) out[no++] = P;
        if (inP != inQ) {
            double r = fP / (fP - fQ);
            wpo_pt I;
            I.s = P.s + (Q.s - P.s) * r;
            I.t = P.t + (Q.t - P.t) * r;
            out[no++] = I;
        }
    }
    return no;
}

/* Structural-nonzero predicate (R6).  Returns 1 and the polygon Pi
 * (nv vertices, counter-clockwise) if the cells overlap with positive measure. */
int wpo_overlap(double a, double b, double c, double d,
                double L1, double U1, double L2, double U2,
                wpo_pt* poly, int* nv_out)
{
    /* energy band  L2^2-U1^2 < h(s,t) = 3/4 (t^2 - s^2) < U2^2-L1^2  */
    double h_lo = L2 * L2 - U1 * U1;
    double h_hi = U2 * U2 - L1 * L1;
    /* (1) box tests, all necessary conditions */
    if (!(0.75 * (d * d - a * a) > h_lo)) return 0;
    if (!(0.75 * (c * c - b * b) < h_hi)) return 0;
    if (!(b + 0.5 * d > L1)) return 0;
    if (!(fmax(a - 0.5 * d, 0.5 * c - b) < U1)) return 0;
    if (!(0.5 * b + d > L2)) return 0;
    if (!(fmax(0.5 * a - d, c - 0.5 * b) < U2)) return 0;
    /* (2) polygon Pi = rectangle clipped by the six half-planes, in order */
    wpo_pt bufA[WPO_MAXV], bufB[WPO_MAXV];
    wpo_pt *cur = bufA, *nxt = bufB;
    int n = 4;
    cur[0].s = a; cur[0].t = c;
    cur[1].s = b; cur[1].t = c;
    cur[2].s = b; cur[2].t = d;
    cur[3].s = a; cur[3].t = d;
    for (int m = 0; m < 6; ++m) {
        n = clip_polygon(cur, n, nxt, m, L1, U1, L2, U2);
        if (n < 3) return 0;
        wpo_pt* tmp = cur; cur = nxt; nxt = tmp;
    }
    /* (3) positive area (shoelace about vertex 0) */
    double area2 = 0.0;
    for (int v = 1; v + 1 < n; ++v) {
        double s1 = cur[v].s - cur[0].s, t1 = cur[v].t - cur[0].t;
        double s2 = cur[v + 1].s - cur[0].s, t2 = cur[v + 1].t - cur[0].t;
        area2 = area2 + (s1 * t2 - s2 * t1);
    }
    if (!(area2 > 0.0)) return 0;
    /* (4) extremes of h on Pi: vertices, plus the two tangent points */
    double hmax = 0.75 * (cur[0].t * cur[0].t - cur[0].s * cur[0].s), hmin = hmax;
    for (int v = 1; v < n; ++v) {
        double h = 0.75 * (cur[v].t * cur[v].t - cur[v].s * cur[v].s);
        hmax = fmax(hmax, h);
        hmin = fmin(hmin, h);
    }
    {   /* minimum of h along q - q'/2 = U1 is at (4U1/3, 2U1/3), h = -U1^2 */
        double s = 4.0 * U1 / 3.0, t = 2.0 * U1 / 3.0;
        if (s >= a && s <= b && t >= c && t <= d
            && halfplane(0, s, t, L1, U1, L2, U2) >= 0.0 && halfplane(2, s, t, L1, U1, L2, U2) >= 0.0
            && halfplane(3, s, t, L1, U1, L2, U2) >= 0.0 && halfplane(4, s, t, L1, U1, L2, U2) >= 0.0
            && halfplane(5, s, t, L1, U1, L2, U2) >= 0.0)
            hmin = fmin(hmin, -(U1 * U1));
    }
    {   /* maximum of h along q' - q/2 = U2 is at (2U2/3, 4U2/3), h = +U2^2 */
        double s = 2.0 * U2 / 3.0, t = 4.0 * U2 / 3.0;
        if (s >= a && s <= b && t >= c && t <= d
            && halfplane(0, s, t, L1, U1, L2, U2) >= 0.0 && halfplane(1, s, t, L1, U1, L2, U2) >= 0.0
            && halfplane(2, s, t, L1, U1, L2, U2) >= 0.0 && halfplane(3, s, t, L1, U1, L2, U2) >= 0.0
            && halfplane(5, s, t, L1, U1, L2, U2) >= 0.0)
            hmax = fmax(hmax, U2 * U2);
    }
    if (!(hmax > h_lo)) return 0;
    if (!(hmin < h_hi)) return 0;
    if (poly) memcpy(poly, cur, (size_t)n * sizeof(wpo_pt));
    if (nv_out) *nv_out = n;
    return 1;
}

/* Geometric pattern.  Row r = (i-1)*n_q + (j-1), column likewise with primes;
 * p has n_p+1 nodes, q has n_q+1.  counts[r] = number of structural nonzeros. */
void wpo_geo_count(int n_p, int n_q, const double* p, const double* q, int32_t* counts)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int r = 0; r < n_p * n_q; ++r) {
        int i = r / n_q, j = r % n_q;
        int32_t cnt = 0;
        for (int ip = 0; ip < n_p; ++ip)
            for (int jp = 0; jp < n_q; ++jp)
                cnt += wpo_overlap(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1], 0, 0);
        counts[r] = cnt;
    }
}

void wpo_geo_fill(int n_p, int n_q, const double* p, const double* q,
                  const int64_t* geo_row_ptr, int32_t* geo_col)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int r = 0; r < n_p * n_q; ++r) {
        int i = r / n_q, j = r % n_q;
        int64_t pos = geo_row_ptr[r];
        for (int ip = 0; ip < n_p; ++ip)
            for (int jp = 0; jp < n_q; ++jp)
                if (wpo_overlap(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1], 0, 0))
                    geo_col[pos++] = ip * n_q + jp;
    }
}

/* Rule R(n) for one geometric element (R7), all coupled pairs at once.
 *   n, xi[n], w[n]      Gauss-Legendre nodes / weights on [-1,1]
 *   n_pairs             coupled channel pairs; pair c has orbital momenta l = pair_l[c]
 *                       (row channel), l' = pair_lp[c] (column channel) and terms
 *                       term_ptr[c] .. term_ptr[c+1]-1, each (k, l1, l1', g)  (A3/A4)
 *   val[c]              matrix element (A15)
 *   absval[c]           the same sum with every term replaced by its modulus (A_e of DESIGN.md R9)
 * Sum over (k,l1,l1') is taken PER NODE, before integrating (R8).
 */
#define WPO_MAXPOW 24
/* Arithmetic type of the rule.  The default build is plain FP64 (the precision the CUDA path is compared with).  With
 * -DWPO_EXTENDED the SAME statements run in long double (x87, 64-bit mantissa): the reference that tells rounding of the
 * FP64 evaluations apart from each other on the ill-conditioned first-bin cells (tests: oracle/perm.py, extended=True).
 * Inputs, Gauss-Legendre nodes and outputs stay double; the predicate and the polygon are the FP64 ones in both builds. */
#ifdef WPO_EXTENDED
typedef long double real;
#define RM(f) f##l
#else
typedef double real;
#define RM(f) f
#endif
static void element_values_inner(double a_, double b_, double c_, double d_,
                                 double L1_, double U1_, double L2_, double U2_,
                                 int n, const double* xi, const double* w, int split,
                                 int n_pairs, const int32_t* pair_l, const int32_t* pair_lp,
                                 const int64_t* term_ptr, const int32_t* term_k, const int32_t* term_l1,
                                 const int32_t* term_l1p, const double* term_g,
                                 real* val, real* absval)
{
    const real a = a_, b = b_, c = c_, d = d_, L1 = L1_, U1 = U1_, L2 = L2_, U2 = U2_;
    wpo_pt poly[WPO_MAXV];
    int nv = 0;
    if (!wpo_overlap(a_, b_, c_, d_, L1_, U1_, L2_, U2_, poly, &nv)) return;
    /* phi-range: angular extent of the polygon Pi (rule R1b) */
    real phi_a = 1e300, phi_b = -1e300;
    for (int v = 0; v < nv; ++v) {
        if (poly[v].s == 0.0 && poly[v].t == 0.0) continue; /* the origin has no angle */
        real ang = RM(atan2)(poly[v].t, poly[v].s);
        phi_a = RM(fmin)(phi_a, ang);
        phi_b = RM(fmax)(phi_b, ang);
    }
    if (!(phi_a < phi_b)) return;
    real norm = 1.0 / RM(sqrt)((U2 - L2) * (b - a) * (U1 - L1) * (d - c)); /* (d_i dbar_j d_i' dbar_j')^{-1/2}, A5/A9 */
    /* Rule R(n): one piece in phi, one piece in u.  Rule RS(n) (split != 0, R14): the phi-range is
     * cut at the rectangle-corner angles where the active member of Lq = max(a/C, c/S) or Uq = min(b/C, d/S)
     * switches (tan phi = c/a, tan phi = d/b), and at every phi-node the u-range is cut at the abscissae where two
     * members of Qmax = min(Uq, U1/zeta1, U2/zeta2) or of Qmin = max(Lq, L1/zeta1, L2/zeta2) of (A14) cross
     * (zeta^2 is linear in u, so each crossing is a closed form); n-point Gauss-Legendre on every piece. */
    real phi_cut[4];
    int n_phi_piece = 1;
    phi_cut[0] = phi_a;
    if (split) {
        real c1 = RM(atan2)(c, a), c2 = RM(atan2)(d, b);
        real lo = RM(fmin)(c1, c2), hi = RM(fmax)(c1, c2);
        if (lo > phi_a && lo < phi_b) phi_cut[n_phi_piece++] = lo;
        if (hi > phi_cut[n_phi_piece - 1] && hi < phi_b) phi_cut[n_phi_piece++] = hi;
    }
    phi_cut[n_phi_piece] = phi_b;
    for (int piece = 0; piece < n_phi_piece; ++piece) {
    real half_phi = 0.5 * (phi_cut[piece + 1] - phi_cut[piece]), mid_phi = 0.5 * (phi_cut[piece] + phi_cut[piece + 1]);
    for (int m = 0; m < n; ++m) {
        real phi = mid_phi + half_phi * xi[m];
        real wphi = half_phi * w[m];
        real C = RM(cos)(phi), S = RM(sin)(phi);
        /* Q-limits from the rectangle, A12 */
        real Lq = RM(fmax)(a / C, c / S), Uq = RM(fmin)(b / C, d / S);
        if (!(Lq < Uq)) continue;
        /* zeta of A11 in the variable u = 1 + x (R7: same rule, conditioned near the
         * pi1 = 0 / pi2 = 0 corners x = -1):  zeta1^2 = b1 + beta u,  zeta2^2 = b2 + beta u */
        real b1 = (C - 0.5 * S) * (C - 0.5 * S);
        real b2 = (0.5 * C - S) * (0.5 * C - S);
        real beta = C * S;
        /* u-support of F > 0 (closed form; zeta^2 linear in u) */
        real u_lo = 0.0, u_hi = 2.0;
        if (L1 > 0.0) u_lo = RM(fmax)(u_lo, ((L1 / Uq) * (L1 / Uq) - b1) / beta);
        if (L2 > 0.0) u_lo = RM(fmax)(u_lo, ((L2 / Uq) * (L2 / Uq) - b2) / beta);
        if (Lq > 0.0) {
            u_hi = RM(fmin)(u_hi, ((U1 / Lq) * (U1 / Lq) - b1) / beta);
            u_hi = RM(fmin)(u_hi, ((U2 / Lq) * (U2 / Lq) - b2) / beta);
        }
        {   /* L1/zeta1 < U2/zeta2  <=>  beta u (L1^2-U2^2) < U2^2 b1 - L1^2 b2 */
            real D = L1 * L1 - U2 * U2, R = U2 * U2 * b1 - L1 * L1 * b2;
            if (D > 0.0) u_hi = RM(fmin)(u_hi, R / (beta * D));
            else if (D < 0.0) u_lo = RM(fmax)(u_lo, R / (beta * D));
            else if (!(0.0 < R)) continue;
        }
        {   /* L2/zeta2 < U1/zeta1  <=>  beta u (L2^2-U1^2) < U1^2 b2 - L2^2 b1 */
            real D = L2 * L2 - U1 * U1, R = U1 * U1 * b2 - L2 * L2 * b1;
            if (D > 0.0) u_hi = RM(fmin)(u_hi, R / (beta * D));
            else if (D < 0.0) u_lo = RM(fmax)(u_lo, R / (beta * D));
            else if (!(0.0 < R)) continue;
        }
        if (!(u_lo < u_hi)) continue;
        real u_cut[8];
        int n_u_piece = 1;
        u_cut[0] = u_lo;
        if (split) {
            real cand[6];
            int nc = 0;
            cand[nc++] = ((U1 / Uq) * (U1 / Uq) - b1) / beta;                         /* Uq = U1/zeta1 */
            cand[nc++] = ((U2 / Uq) * (U2 / Uq) - b2) / beta;                         /* Uq = U2/zeta2 */
            if (U1 != U2) cand[nc++] = (U2 * U2 * b1 - U1 * U1 * b2) / (beta * (U1 * U1 - U2 * U2)); /* U1/zeta1 = U2/zeta2 */
            if (Lq > 0.0) {
                cand[nc++] = ((L1 / Lq) * (L1 / Lq) - b1) / beta;                     /* Lq = L1/zeta1 */
                cand[nc++] = ((L2 / Lq) * (L2 / Lq) - b2) / beta;                     /* Lq = L2/zeta2 */
            }
            if (L1 != L2) cand[nc++] = (L2 * L2 * b1 - L1 * L1 * b2) / (beta * (L1 * L1 - L2 * L2)); /* L1/zeta1 = L2/zeta2 */
            for (int i1 = 1; i1 < nc; ++i1) {                                         /* ascending */
                real key = cand[i1];
                int i0 = i1 - 1;
                while (i0 >= 0 && cand[i0] > key) { cand[i0 + 1] = cand[i0]; --i0; }
                cand[i0 + 1] = key;
            }
            for (int i1 = 0; i1 < nc; ++i1)
                if (cand[i1] > u_cut[n_u_piece - 1] && cand[i1] < u_hi) u_cut[n_u_piece++] = cand[i1];
        }
        u_cut[n_u_piece] = u_hi;
        /* powers of cos, sin */
        real cp[WPO_MAXPOW], sp[WPO_MAXPOW];
        cp[0] = 1.0; sp[0] = 1.0;
        for (int e = 1; e < WPO_MAXPOW; ++e) { cp[e] = cp[e - 1] * C; sp[e] = sp[e - 1] * S; }
        for (int upiece = 0; upiece < n_u_piece; ++upiece) {
        real half_u = 0.5 * (u_cut[upiece + 1] - u_cut[upiece]), mid_u = 0.5 * (u_cut[upiece] + u_cut[upiece + 1]);
        if (split == 2) {
            /* Rule RA(n) (R15), s-wave term only (k = l1 = l1' = 0, l = l' = 0): on a piece between two
             * cuts the active members of (A14)'s min and max do not change, each is a constant or a constant over
             * zeta^2, so with F = 1/2 (Qmax^2 - Qmin^2) = 1/2 (dA + dB / zeta1^2 + dC / zeta2^2) the u-integral of
             * F / (zeta1 zeta2) is elementary:
             *   I0 = int du / (zeta1 zeta2)     = (2/beta) ln[(zeta1h + zeta2h) / (zeta1l + zeta2l)]
             *   I1 = int du / (zeta1^3 zeta2)   = (2/beta) (1/zeta1l^2 - 1/zeta1h^2) / (zeta2h/zeta1h + zeta2l/zeta1l)
             *   I2 = int du / (zeta1 zeta2^3)   = (2/beta) (1/zeta2l^2 - 1/zeta2h^2) / (zeta1h/zeta2h + zeta1l/zeta2l)
             * (l, h = lower, upper end of the piece; the forms for I1, I2 have no cancellation when b1 -> b2).
             * The active members are read off at the midpoint of the piece. */
            real ul = u_cut[upiece], uh = u_cut[upiece + 1];
            real z1m = RM(sqrt)(b1 + beta * mid_u), z2m = RM(sqrt)(b2 + beta * mid_u);
            real dA = 0.0, dB = 0.0, dC = 0.0;
            {   /* Qmax^2 = min(Uq^2, U1^2/zeta1^2, U2^2/zeta2^2) */
                real m0 = Uq, m1 = U1 / z1m, m2 = U2 / z2m;
                if (m0 <= m1 && m0 <= m2) dA += Uq * Uq; else if (m1 <= m2) dB += U1 * U1; else dC += U2 * U2;
            }
            {   /* Qmin^2 = max(Lq^2, L1^2/zeta1^2, L2^2/zeta2^2) */
                real m0 = Lq, m1 = L1 / z1m, m2 = L2 / z2m;
                if (m0 >= m1 && m0 >= m2) dA -= Lq * Lq; else if (m1 >= m2) dB -= L1 * L1; else dC -= L2 * L2;
            }
            real z1l = RM(sqrt)(b1 + beta * ul), z2l = RM(sqrt)(b2 + beta * ul);
            real z1h = RM(sqrt)(b1 + beta * uh), z2h = RM(sqrt)(b2 + beta * uh);
            /* differences of the ends written without cancellation: zeta_h - zeta_l = beta du / (zeta_h + zeta_l),
             * 1/zeta_l^2 - 1/zeta_h^2 = beta du / (zeta_l^2 zeta_h^2) */
            real du = uh - ul;
            real integral = 0.0;
            if (dA != 0.0)
                integral += dA * (2.0 / beta) * RM(log1p)((beta * du / (z1h + z1l) + beta * du / (z2h + z2l)) / (z1l + z2l));
            if (dB != 0.0) integral += dB * 2.0 * du / (z1l * z1l * z1h * z1h) / (z2h / z1h + z2l / z1l);
            if (dC != 0.0) integral += dC * 2.0 * du / (z2l * z2l * z2h * z2h) / (z1h / z2h + z1l / z2l);
            if (integral > 0.0) {
                for (int cidx = 0; cidx < n_pairs; ++cidx) {
                    real g = term_g[term_ptr[cidx]];
                    val[cidx] += wphi * 0.5 * integral * g * C * S;
                    absval[cidx] += wphi * 0.5 * integral * RM(fabs)(g) * C * S;
                }
            }
            continue;
        }
        for (int r = 0; r < n; ++r) {
            real u = mid_u + half_u * xi[r];
            real x = u - 1.0;
            real wx = half_u * w[r];
            real zeta1 = RM(sqrt)(b1 + beta * u), zeta2 = RM(sqrt)(b2 + beta * u);
            /* F of A14, clamped (R5) */
            real Qmax = RM(fmin)(RM(fmin)(Uq, U1 / zeta1), U2 / zeta2);
            real Qmin = RM(fmax)(RM(fmax)(Lq, L1 / zeta1), L2 / zeta2);
            if (!(Qmax > Qmin)) continue;
            real F = 0.5 * (Qmax * Qmax - Qmin * Qmin);
            /* Legendre polynomials by the three-term recurrence */
            real P[WPO_MAXPOW];
            P[0] = 1.0; P[1] = x;
            for (int k = 2; k < WPO_MAXPOW; ++k) P[k] = ((2 * k - 1) * x * P[k - 1] - (k - 1) * P[k - 2]) / k;
            real z1p[WPO_MAXPOW], z2p[WPO_MAXPOW]; /* zeta^m */
            z1p[0] = 1.0; z2p[0] = 1.0;
            for (int e = 1; e < WPO_MAXPOW; ++e) { z1p[e] = z1p[e - 1] * zeta1; z2p[e] = z2p[e - 1] * zeta2; }
            real wF = wphi * wx * F;
            for (int cidx = 0; cidx < n_pairs; ++cidx) {
                int l = pair_l[cidx], lp = pair_lp[cidx];
                real sum = 0.0, asum = 0.0;
                for (int64_t tt = term_ptr[cidx]; tt < term_ptr[cidx + 1]; ++tt) {
                    int l1 = term_l1[tt], l1p = term_l1p[tt];
                    int A = l1 + l1p;                 /* power of q  = Q RM(cos)(phi) (R1) */
                    int B = (l - l1) + (lp - l1p);    /* power of q' = Q RM(sin)(phi) */
                    real term = term_g[tt] * P[term_k[tt]] * cp[A + 1] * sp[B + 1];
                    sum += term;
                    asum += RM(fabs)(term);
                }
                real denom = z1p[lp + 1] * z2p[l + 1];
                val[cidx] += wF * sum / denom;
                absval[cidx] += wF * asum / denom;
            }
        }
        } /* u pieces */
    }
    } /* phi pieces */
    for (int cidx = 0; cidx < n_pairs; ++cidx) { val[cidx] *= norm; absval[cidx] *= norm; }
}


static void element_values(double a, double b, double c, double d,
                           double L1, double U1, double L2, double U2,
                           int n, const double* xi, const double* w, int split,
                           int n_pairs, const int32_t* pair_l, const int32_t* pair_lp,
                           const int64_t* term_ptr, const int32_t* term_k, const int32_t* term_l1,
                           const int32_t* term_l1p, const double* term_g,
                           double* val_out, double* absval_out)
{
    for (int cidx = 0; cidx < n_pairs; ++cidx) { val_out[cidx] = 0.0; absval_out[cidx] = 0.0; }
    real* val = (real*)calloc(2 * (size_t)n_pairs, sizeof(real));   /* the sums are kept in the rule's arithmetic type */
    real* absval = val + n_pairs;
    element_values_inner(a, b, c, d, L1, U1, L2, U2, n, xi, w, split, n_pairs, pair_l, pair_lp, term_ptr, term_k, term_l1, term_l1p, term_g,
                         val, absval);
    for (int cidx = 0; cidx < n_pairs; ++cidx) { val_out[cidx] = (double)val[cidx]; absval_out[cidx] = (double)absval[cidx]; }
    free(val);
}

/* Values of n_elem listed geometric elements (row cell (ei,ej), column cell (eip,ejp),
 * all 0-based bin indices).  val/absval are [n_elem][n_pairs], row-major. */
void wpo_elements_rule(int n_p, int n_q, const double* p, const double* q,
                       int64_t n_elem, const int32_t* ei, const int32_t* ej, const int32_t* eip, const int32_t* ejp,
                       int n, const double* xi, const double* w, int split,
                       int n_pairs, const int32_t* pair_l, const int32_t* pair_lp,
                       const int64_t* term_ptr, const int32_t* term_k, const int32_t* term_l1,
                       const int32_t* term_l1p, const double* term_g,
                       double* val, double* absval)
{
    (void)n_p; (void)n_q;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t e = 0; e < n_elem; ++e) {
        int i = ei[e], j = ej[e], ip = eip[e], jp = ejp[e];
        element_values(q[j], q[j + 1], q[jp], q[jp + 1], p[ip], p[ip + 1], p[i], p[i + 1],
                       n, xi, w, split, n_pairs, pair_l, pair_lp, term_ptr, term_k, term_l1, term_l1p, term_g,
                       val + e * n_pairs, absval + e * n_pairs);
    }
}

/* rule R(n) */
void wpo_elements(int n_p, int n_q, const double* p, const double* q,
                  int64_t n_elem, const int32_t* ei, const int32_t* ej, const int32_t* eip, const int32_t* ejp,
                  int n, const double* xi, const double* w,
                  int n_pairs, const int32_t* pair_l, const int32_t* pair_lp,
                  const int64_t* term_ptr, const int32_t* term_k, const int32_t* term_l1,
                  const int32_t* term_l1p, const double* term_g,
                  double* val, double* absval)
{
    wpo_elements_rule(n_p, n_q, p, q, n_elem, ei, ej, eip, ejp, n, xi, w, 0, n_pairs, pair_l, pair_lp, term_ptr, term_k, term_l1,
                      term_l1p, term_g, val, absval);
}

/* y = P0 x, CSR, each row summed sequentially in column order. */
void wpo_spmv(int64_t rows, const int64_t* row_ptr, const int32_t* col_idx, const double* values,
              const double* x, double* y)
{
    for (int64_t r = 0; r < rows; ++r) {
        double acc = 0.0;
        for (int64_t e = row_ptr[r]; e < row_ptr[r + 1]; ++e) acc += values[e] * x[col_idx[e]];
        y[r] = acc;
    }
}

int wpo_num_threads(void)
{
    int nt = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        nt = omp_get_num_threads();
    }
#endif
    return nt;
}
