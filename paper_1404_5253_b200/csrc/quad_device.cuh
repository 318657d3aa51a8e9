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
