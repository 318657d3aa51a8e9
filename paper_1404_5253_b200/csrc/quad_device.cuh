// quad_device.cuh -- device pieces of the quadrature rule R(n) (R7) for (A15)
// with F of (A14), zeta of (A11) and the
// Q-limits of (A12).  Product path; FMA contraction allowed here.
#pragma once
#include <cuda_runtime.h>

namespace wpcd_quad {

struct Cell { double a, b, c, d, L1, U1, L2, U2; };

struct PhiNode {
    double C, S;          // cos(phi), sin(phi)
    double Lq, Uq;        // Q-limits from the (q,q') rectangle, (A12)
    double b1, b2, beta;  // zeta1^2 = b1 + beta u, zeta2^2 = b2 + beta u, u = 1 + x, (A11)
    double u_lo, u_hi;    // closed-form support of F > 0 in u
};

// Everything of R(n) that depends on phi only.  Returns false when the node contributes 0.
__device__ __forceinline__ bool phi_node(const Cell& z, double phi, PhiNode& s)
{
    sincos(phi, &s.S, &s.C);
    s.Lq = fmax(z.a / s.C, z.c / s.S);
    s.Uq = fmin(z.b / s.C, z.d / s.S);
    if (!(s.Lq < s.Uq)) return false;
    {   // (A11) in u = 1 + x: b1 = (C - S/2)^2, b2 = (C/2 - S)^2 -- no cancellation near x = -1
        double d1 = s.C - 0.5 * s.S, d2 = 0.5 * s.C - s.S;
        s.b1 = d1 * d1; s.b2 = d2 * d2;
    }
    s.beta = s.C * s.S;
    double u_lo = 0.0, u_hi = 2.0;
    if (z.L1 > 0.0) { double r = z.L1 / s.Uq; u_lo = fmax(u_lo, (r * r - s.b1) / s.beta); }
    if (z.L2 > 0.0) { double r = z.L2 / s.Uq; u_lo = fmax(u_lo, (r * r - s.b2) / s.beta); }
    if (s.Lq > 0.0) {
        double r1 = z.U1 / s.Lq, r2 = z.U2 / s.Lq;
        u_hi = fmin(u_hi, (r1 * r1 - s.b1) / s.beta);
        u_hi = fmin(u_hi, (r2 * r2 - s.b2) / s.beta);
    }
    {   // L1/zeta1 < U2/zeta2  <=>  beta u (L1^2-U2^2) < U2^2 b1 - L1^2 b2.  The sign of D must be
        // decided on unfused products (exact ties L1 == U2 are systematic on p == q grids).
        double D = __dsub_rn(__dmul_rn(z.L1, z.L1), __dmul_rn(z.U2, z.U2));
        double R = z.U2 * z.U2 * s.b1 - z.L1 * z.L1 * s.b2;
        if (D > 0.0) u_hi = fmin(u_hi, R / (s.beta * D));
        else if (D < 0.0) u_lo = fmax(u_lo, R / (s.beta * D));
        else if (!(0.0 < R)) return false;
    }
    {   // L2/zeta2 < U1/zeta1  <=>  beta u (L2^2-U1^2) < U1^2 b2 - L2^2 b1
        double D = __dsub_rn(__dmul_rn(z.L2, z.L2), __dmul_rn(z.U1, z.U1));
        double R = z.U1 * z.U1 * s.b2 - z.L2 * z.L2 * s.b1;
        if (D > 0.0) u_hi = fmin(u_hi, R / (s.beta * D));
        else if (D < 0.0) u_lo = fmax(u_lo, R / (s.beta * D));
        else if (!(0.0 < R)) return false;
    }
    s.u_lo = u_lo; s.u_hi = u_hi;
    return u_lo < u_hi;
}

// F of (A14), clamped at 0 (R5), from 1/zeta1, 1/zeta2.
__device__ __forceinline__ double F_A14(const Cell& z, const PhiNode& s, double iz1, double iz2)
{
    double Qmax = fmin(fmin(s.Uq, z.U1 * iz1), z.U2 * iz2);
    double Qmin = fmax(fmax(s.Lq, z.L1 * iz1), z.L2 * iz2);
    return Qmax > Qmin ? 0.5 * (Qmax - Qmin) * (Qmax + Qmin) : 0.0;
}

// ---- the same rule in squared variables (no square roots, one reciprocal per limit).
// Q-limits enter (A14) only through their squares: F = 1/2 (min Q^2 - max Q^2), and squaring is
// monotone on Q >= 0, so F needs 1/zeta^2 only; u-limits need (L/U_q)^2 = L^2 / U_q^2.
struct CellSq { double a2, b2, c2, d2, L1s, U1s, L2s, U2s; };

__device__ __forceinline__ CellSq square_cell(const Cell& z)
{
    CellSq s;
    s.a2 = z.a * z.a; s.b2 = z.b * z.b; s.c2 = z.c * z.c; s.d2 = z.d * z.d;
    s.L1s = z.L1 * z.L1; s.U1s = z.U1 * z.U1; s.L2s = z.L2 * z.L2; s.U2s = z.U2 * z.U2;
    return s;
}

struct PhiNodeSq {
    double C, S;
    double Lq2, Uq2;      // squares of the Q-limits of (A12)
    double b1, b2, beta;
    double u_lo, u_hi;
    double ibeta;         // 1/beta
};

__device__ __forceinline__ bool phi_node_sq(const Cell& z, const CellSq& zs, double phi, PhiNodeSq& s)
{
    sincos(phi, &s.S, &s.C);
    const double C2 = s.C * s.C, S2 = s.S * s.S;
    s.beta = s.C * s.S;
    const double ib2 = __drcp_rn(C2 * S2);          // 1/beta^2  ->  1/C^2 = S^2 ib2, 1/S^2 = C^2 ib2, 1/beta = beta ib2
    const double iC2 = S2 * ib2, iS2 = C2 * ib2, ibeta = s.beta * ib2;
    s.Lq2 = fmax(zs.a2 * iC2, zs.c2 * iS2);
    s.Uq2 = fmin(zs.b2 * iC2, zs.d2 * iS2);
    if (!(s.Lq2 < s.Uq2)) return false;
    {
        const double d1 = s.C - 0.5 * s.S, d2 = 0.5 * s.C - s.S;
        s.b1 = d1 * d1; s.b2 = d2 * d2;
    }
    double u_lo = 0.0, u_hi = 2.0;
    if (z.L1 > 0.0 || z.L2 > 0.0) {
        const double iUq2 = __drcp_rn(s.Uq2);
        if (z.L1 > 0.0) u_lo = fmax(u_lo, (zs.L1s * iUq2 - s.b1) * ibeta);
        if (z.L2 > 0.0) u_lo = fmax(u_lo, (zs.L2s * iUq2 - s.b2) * ibeta);
    }
    if (s.Lq2 > 0.0) {
        const double iLq2 = __drcp_rn(s.Lq2);
        u_hi = fmin(u_hi, (zs.U1s * iLq2 - s.b1) * ibeta);
        u_hi = fmin(u_hi, (zs.U2s * iLq2 - s.b2) * ibeta);
    }
    {   // L1/zeta1 < U2/zeta2  <=>  beta u (L1^2-U2^2) < U2^2 b1 - L1^2 b2; sign of D on unfused products
        const double D = __dsub_rn(__dmul_rn(z.L1, z.L1), __dmul_rn(z.U2, z.U2));
        const double R = zs.U2s * s.b1 - zs.L1s * s.b2;
        if (D > 0.0) u_hi = fmin(u_hi, R * ibeta / D);
        else if (D < 0.0) u_lo = fmax(u_lo, R * ibeta / D);
        else if (!(0.0 < R)) return false;
    }
    {   // L2/zeta2 < U1/zeta1  <=>  beta u (L2^2-U1^2) < U1^2 b2 - L2^2 b1
        const double D = __dsub_rn(__dmul_rn(z.L2, z.L2), __dmul_rn(z.U1, z.U1));
        const double R = zs.U1s * s.b2 - zs.L2s * s.b1;
        if (D > 0.0) u_hi = fmin(u_hi, R * ibeta / D);
        else if (D < 0.0) u_lo = fmax(u_lo, R * ibeta / D);
        else if (!(0.0 < R)) return false;
    }
    s.u_lo = u_lo; s.u_hi = u_hi; s.ibeta = ibeta;
    return u_lo < u_hi;
}

// 2 F of (A14) from r1 = 1/zeta1^2, r2 = 1/zeta2^2 (clamped at 0, R5)
__device__ __forceinline__ double twoF_A14_sq(const CellSq& zs, const PhiNodeSq& s, double r1, double r2)
{
    // plain compare-and-select (all operands are finite here; fmin/fmax would add NaN handling)
    const double pU1 = zs.U1s * r1, pU2 = zs.U2s * r2, pL1 = zs.L1s * r1, pL2 = zs.L2s * r2;
    double Qmax2 = pU1 < s.Uq2 ? pU1 : s.Uq2;
    Qmax2 = pU2 < Qmax2 ? pU2 : Qmax2;
    double Qmin2 = pL1 > s.Lq2 ? pL1 : s.Lq2;
    Qmin2 = pL2 > Qmin2 ? pL2 : Qmin2;
    const double F2 = Qmax2 - Qmin2;
    return F2 > 0.0 ? F2 : 0.0;
}

// ---- kink-split rule RS(n) (R14): cuts of the phi-range and of the u-range.
constexpr int SPLIT_MAX_PHI = 3;   // pieces in phi
constexpr int SPLIT_MAX_U = 7;     // pieces in u

// cut[0 .. n_piece]: the range (phi_a, phi_b) cut at the rectangle-corner angles atan2(c, a), atan2(d, b) inside it
// (static indexing only: the array stays in registers).
__device__ __forceinline__ int split_phi(const Cell& z, double phi_a, double phi_b, double (&cut)[SPLIT_MAX_PHI + 1])
{
    const double c1 = atan2(z.c, z.a), c2 = atan2(z.d, z.b);
    const double lo = fmin(c1, c2), hi = fmax(c1, c2);
    const bool lo_in = lo > phi_a && lo < phi_b;
    const double last = lo_in ? lo : phi_a;
    const bool hi_in = hi > last && hi < phi_b;
    cut[0] = phi_a;
    cut[1] = lo_in ? lo : (hi_in ? hi : phi_b);
    cut[2] = (lo_in && hi_in) ? hi : phi_b;
    cut[3] = phi_b;
    return 1 + (lo_in ? 1 : 0) + (hi_in ? 1 : 0);
}

// The six candidate cuts of the u-range, ascending (+inf where a crossing does not exist): crossings of the members of
// Qmax = min(Uq, U1/zeta1, U2/zeta2) and of Qmin = max(Lq, L1/zeta1, L2/zeta2) (zeta^2 linear in u: closed forms).
// The pieces are (u_lo, c_1), (c_1, c_2), ..., (c_k, u_hi) over the candidates strictly inside, taken in order:
//   lower = u_lo;  for each c: if (c > lower && c < u_hi) { piece(lower, c); lower = c; }  piece(lower, u_hi).
__device__ __forceinline__ void split_u_candidates(const Cell& z, const CellSq& zs, const PhiNodeSq& s, double (&cand)[6])
{
    const double inf = __longlong_as_double(0x7ff0000000000000ll);
    const double iUq2 = __drcp_rn(s.Uq2);
    cand[0] = (zs.U1s * iUq2 - s.b1) * s.ibeta;                                                      // Uq = U1/zeta1
    cand[1] = (zs.U2s * iUq2 - s.b2) * s.ibeta;                                                      // Uq = U2/zeta2
    cand[2] = z.U1 != z.U2 ? (zs.U2s * s.b1 - zs.U1s * s.b2) * s.ibeta / (zs.U1s - zs.U2s) : inf;     // U1/zeta1 = U2/zeta2
    if (s.Lq2 > 0.0) {
        const double iLq2 = __drcp_rn(s.Lq2);
        cand[3] = (zs.L1s * iLq2 - s.b1) * s.ibeta;                                                  // Lq = L1/zeta1
        cand[4] = (zs.L2s * iLq2 - s.b2) * s.ibeta;                                                  // Lq = L2/zeta2
    } else {
        cand[3] = inf; cand[4] = inf;
    }
    cand[5] = z.L1 != z.L2 ? (zs.L2s * s.b1 - zs.L1s * s.b2) * s.ibeta / (zs.L1s - zs.L2s) : inf;     // L1/zeta1 = L2/zeta2
    // ascending: odd-even transposition network on six registers
#pragma unroll
    for (int pass = 0; pass < 6; ++pass) {
#pragma unroll
        for (int i = pass & 1; i + 1 < 6; i += 2) {
            const double lo = fmin(cand[i], cand[i + 1]), hi = fmax(cand[i], cand[i + 1]);
            cand[i] = lo; cand[i + 1] = hi;
        }
    }
}

__device__ __forceinline__ Cell load_cell(const double* __restrict__ p, const double* __restrict__ q, int n_q, int row, int col)
{
    int i = row / n_q, j = row - i * n_q;
    int ip = col / n_q, jp = col - ip * n_q;
    Cell z;
    z.a = q[j]; z.b = q[j + 1]; z.c = q[jp]; z.d = q[jp + 1];
    z.L1 = p[ip]; z.U1 = p[ip + 1]; z.L2 = p[i]; z.U2 = p[i + 1];
    return z;
}

__device__ __forceinline__ double cell_norm(const Cell& z)
{
    return rsqrt((z.U2 - z.L2) * (z.b - z.a) * (z.U1 - z.L1) * (z.d - z.c));   // (A5)/(A9)
}

}  // namespace wpcd_quad
