// fill.cu -- "calculation of the nonzero elements of P0" (paper step 3):
// FP64 Gauss-Legendre quadrature of (A15) over the clipped overlap region.
//
// This file: the s-wave path (configs 1-2: one channel, one term).  LPE lanes share one element,
// each lane owns whole phi-nodes and runs the inner x-rule in squared variables (one rsqrt per
// node); shuffles reduce.  The coupled-channel path (configs 3-5) is fill_coupled.cu.
#include <math.h>
#include <stdlib.h>

#include "quad_device.cuh"
#include "wpcd_internal.h"

using namespace wpcd_quad;
using wpcd_detail::QuadRule;

namespace {

// The rule travels as a by-value __grid_constant__ kernel parameter (wpcd_internal.h QuadRule): it sits in the
// launch's own constant bank, so builds with different orders may overlap on one device (streams or threads), and
// with a compile-time order the nodes and weights still fold into constant-bank operands.

// ------------------------------------------------------------------ s-wave
// NQ > 0: rule order fixed at compile time (loops unrolled, nodes and weights become immediates
// of the constant bank); NQ = 0: any order.
template <int LPE, int NQ>
__global__ void __launch_bounds__(256)
fill_swave_kernel(const __grid_constant__ QuadRule rule, const double* __restrict__ p, const double* __restrict__ q, int n_q, int n_rt, double g0,
                  int64_t nnz_geo, const int32_t* __restrict__ geo_col, const int32_t* __restrict__ geo_row,
                  const double2* __restrict__ geo_phi, int32_t* __restrict__ col_idx, double* __restrict__ values)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t e = t / LPE;
    const int sub = (int)(t - e * LPE);
    const bool valid = e < nnz_geo;
    const int n = NQ > 0 ? NQ : n_rt;
    double acc = 0.0;
    double norm = 0.0;
    int col = 0;
    if (valid) {
        col = geo_col[e];
        const int row = geo_row[e];
        const double2 ph = geo_phi[e];
        const Cell z = load_cell(p, q, n_q, row, col);
        const CellSq zs = square_cell(z);
        norm = cell_norm(z);
        const double half_phi = 0.5 * (ph.y - ph.x), mid_phi = 0.5 * (ph.x + ph.y);
        if (ph.x < ph.y) {
#pragma unroll 1
            for (int m = sub; m < n; m += LPE) {
                PhiNodeSq s;
                if (!phi_node_sq(z, zs, mid_phi + half_phi * rule.xi[m], s)) continue;
                const double half_u = 0.5 * (s.u_hi - s.u_lo), mid_u = 0.5 * (s.u_lo + s.u_hi);
                double inner = 0.0;
#pragma unroll
                for (int r = 0; r < n; ++r) {
                    const double u = mid_u + half_u * rule.xi[r];
                    const double z1 = s.b1 + s.beta * u, z2 = s.b2 + s.beta * u;    // zeta1^2, zeta2^2 (A11)
                    const double t = rsqrt(z1 * z2);                                // 1/(zeta1 zeta2)
                    const double t2 = t * t;
                    inner += rule.w[r] * twoF_A14_sq(zs, s, t2 * z2, t2 * z1) * t;
                }
                acc += half_phi * rule.w[m] * half_u * s.beta * inner;    // cos*sin = beta
            }
        }
    }
#pragma unroll
    for (int o = LPE / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (valid && sub == 0) {
        values[e] = 0.5 * g0 * norm * acc;    // the 1/2 of (A14)
        col_idx[e] = col;
    }
}

// ------------------------------------------------------------------ s-wave, kink-split rule RS(n) (R14)
// The work items of an element are its (phi-piece, phi-node) pairs, dealt to the LPE lanes; each item integrates its
// u-pieces one after the other (sorted candidate cuts in registers, no arrays).
template <int LPE, int NQ>
__global__ void __launch_bounds__(256)
fill_swave_split_kernel(const __grid_constant__ QuadRule rule, const double* __restrict__ p, const double* __restrict__ q, int n_q, int n_rt, double g0,
                        int64_t nnz_geo, const int32_t* __restrict__ geo_col, const int32_t* __restrict__ geo_row,
                        const double2* __restrict__ geo_phi, int32_t* __restrict__ col_idx, double* __restrict__ values)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t e = t / LPE;
    const int sub = (int)(t - e * LPE);
    const bool valid = e < nnz_geo;
    const int n = NQ > 0 ? NQ : n_rt;
    double acc = 0.0;
    double norm = 0.0;
    int col = 0;
    if (valid) {
        col = geo_col[e];
        const int row = geo_row[e];
        const double2 ph = geo_phi[e];
        const Cell z = load_cell(p, q, n_q, row, col);
        const CellSq zs = square_cell(z);
        norm = cell_norm(z);
        if (ph.x < ph.y) {
            double pc[SPLIT_MAX_PHI + 1];
            const int n_piece = split_phi(z, ph.x, ph.y, pc);
#pragma unroll 1
            for (int item = sub; item < n_piece * n; item += LPE) {
                const int piece = item / n, m = item - piece * n;
                const double pa = piece == 0 ? pc[0] : (piece == 1 ? pc[1] : pc[2]);
                const double pb = piece == 0 ? pc[1] : (piece == 1 ? pc[2] : pc[3]);
                const double half_phi = 0.5 * (pb - pa), mid_phi = 0.5 * (pa + pb);
                PhiNodeSq s;
                if (!phi_node_sq(z, zs, mid_phi + half_phi * rule.xi[m], s)) continue;
                double cand[6];
                split_u_candidates(z, zs, s, cand);
                auto piece_sum = [&](double lo, double hi) {
                    const double half_u = 0.5 * (hi - lo), mid_u = 0.5 * (lo + hi);
                    double inner = 0.0;
#pragma unroll
                    for (int r = 0; r < n; ++r) {
                        const double u = mid_u + half_u * rule.xi[r];
                        const double z1 = s.b1 + s.beta * u, z2 = s.b2 + s.beta * u;    // zeta1^2, zeta2^2 (A11)
                        const double t = rsqrt(z1 * z2);                                // 1/(zeta1 zeta2)
                        const double t2 = t * t;
                        inner += rule.w[r] * twoF_A14_sq(zs, s, t2 * z2, t2 * z1) * t;
                    }
                    return half_u * inner;
                };
                // cut list in local memory (8 doubles, L1-resident): one copy of the inner rule instead of seven
                double cut[SPLIT_MAX_U + 1];
                int np = 1;
                cut[0] = s.u_lo;
#pragma unroll
                for (int i = 0; i < 6; ++i) {
                    if (cand[i] > cut[np - 1] && cand[i] < s.u_hi) cut[np++] = cand[i];
                }
                cut[np] = s.u_hi;
                double node = 0.0;
#pragma unroll 1
                for (int k = 0; k < np; ++k) node += piece_sum(cut[k], cut[k + 1]);
                acc += half_phi * rule.w[m] * s.beta * node;    // cos*sin = beta
            }
        }
    }
#pragma unroll
    for (int o = LPE / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (valid && sub == 0) {
        values[e] = 0.5 * g0 * norm * acc;    // the 1/2 of (A14)
        col_idx[e] = col;
    }
}

// ------------------------------------------------------------------ s-wave, rule RA(n): exact u-integral (R15)
// Same work items and cuts as the kink-split kernel; on a piece the active members of (A14)'s min / max are fixed, so
// int 2F / (zeta1 zeta2) du = dA I0 + dB I1 + dC I2 in closed form (squared variables, one division per term,
// end-point square roots carried from piece to piece).
template <int LPE>
__global__ void __launch_bounds__(256)
fill_swave_analytic_kernel(const __grid_constant__ QuadRule rule, const double* __restrict__ p, const double* __restrict__ q, int n_q, int n, double g0,
                           int64_t nnz_geo, const int32_t* __restrict__ geo_col, const int32_t* __restrict__ geo_row,
                           const double2* __restrict__ geo_phi, int32_t* __restrict__ col_idx, double* __restrict__ values)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t e = t / LPE;
    const int sub = (int)(t - e * LPE);
    const bool valid = e < nnz_geo;
    double acc = 0.0;
    double norm = 0.0;
    int col = 0;
    if (valid) {
        col = geo_col[e];
        const int row = geo_row[e];
        const double2 ph = geo_phi[e];
        const Cell z = load_cell(p, q, n_q, row, col);
        const CellSq zs = square_cell(z);
        norm = cell_norm(z);
        if (ph.x < ph.y) {
            double pc[SPLIT_MAX_PHI + 1];
            const int n_piece = split_phi(z, ph.x, ph.y, pc);
#pragma unroll 1
            for (int item = sub; item < n_piece * n; item += LPE) {
                const int piece = item / n, m = item - piece * n;
                const double pa = piece == 0 ? pc[0] : (piece == 1 ? pc[1] : pc[2]);
                const double pb = piece == 0 ? pc[1] : (piece == 1 ? pc[2] : pc[3]);
                const double half_phi = 0.5 * (pb - pa), mid_phi = 0.5 * (pa + pb);
                PhiNodeSq s;
                if (!phi_node_sq(z, zs, mid_phi + half_phi * rule.xi[m], s)) continue;
                double cand[6];
                split_u_candidates(z, zs, s, cand);
                double cut[SPLIT_MAX_U + 1];
                int np = 1;
                cut[0] = s.u_lo;
#pragma unroll
                for (int i = 0; i < 6; ++i) {
                    if (cand[i] > cut[np - 1] && cand[i] < s.u_hi) cut[np++] = cand[i];
                }
                cut[np] = s.u_hi;
                double node = 0.0;
                double z1l = sqrt(s.b1 + s.beta * cut[0]), z2l = sqrt(s.b2 + s.beta * cut[0]);
#pragma unroll 1
                for (int k = 0; k < np; ++k) {
                    const double ul = cut[k], uh = cut[k + 1], du = uh - ul;
                    const double um = 0.5 * (ul + uh);
                    const double z1m2 = s.b1 + s.beta * um, z2m2 = s.b2 + s.beta * um;     // zeta^2 at the midpoint
                    const double z1h = sqrt(s.b1 + s.beta * uh), z2h = sqrt(s.b2 + s.beta * uh);
                    // active member of Qmax^2 = min(Uq^2, U1^2/zeta1^2, U2^2/zeta2^2) and of Qmin^2 = max(Lq^2, L1^2/.., L2^2/..)
                    double dA = 0.0, dB = 0.0, dC = 0.0;
                    if (s.Uq2 * z1m2 <= zs.U1s && s.Uq2 * z2m2 <= zs.U2s) dA = s.Uq2;
                    else if (zs.U1s * z2m2 <= zs.U2s * z1m2) dB = zs.U1s;
                    else dC = zs.U2s;
                    if (s.Lq2 * z1m2 >= zs.L1s && s.Lq2 * z2m2 >= zs.L2s) dA -= s.Lq2;
                    else if (zs.L1s * z2m2 >= zs.L2s * z1m2) dB -= zs.L1s;
                    else dC -= zs.L2s;
                    double integral = 0.0;
                    const double bdu = s.beta * du;
                    if (dA != 0.0) {
                        const double s1 = z1h + z1l, s2 = z2h + z2l;
                        integral += dA * 2.0 * s.ibeta * log1p(bdu * (s1 + s2) / (s1 * s2 * (z1l + z2l)));
                    }
                    if (dB != 0.0) integral += dB * 2.0 * du / (z1l * z1h * (z2h * z1l + z2l * z1h));
                    if (dC != 0.0) integral += dC * 2.0 * du / (z2l * z2h * (z1h * z2l + z1l * z2h));
                    if (integral > 0.0) node += integral;
                    z1l = z1h; z2l = z2h;
                }
                acc += half_phi * rule.w[m] * s.beta * node;    // cos*sin = beta
            }
        }
    }
#pragma unroll
    for (int o = LPE / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (valid && sub == 0) {
        values[e] = 0.5 * g0 * norm * acc;    // the 1/2 of (A14)
        col_idx[e] = col;
    }
}

}  // namespace

namespace wpcd_detail {

cudaError_t launch_fill_swave(const wpcd_grid* g, const wpcd_channels* ch, int n_quad, int rule, const QuadRule& qr,
                              int64_t nnz_geo, const Workspace& ws, int32_t* col_idx, double* values, cudaStream_t st)
{
    if (nnz_geo == 0) return cudaSuccess;
    // lanes per element: whole phi-nodes per lane, no idle lanes when n is a multiple of LPE
    int lpe = (n_quad % 8 == 0) ? 8 : (n_quad % 4 == 0) ? 4 : (n_quad % 2 == 0) ? 2 : 1;
    int64_t threads = nnz_geo * lpe;
    int blocks = (int)((threads + 255) / 256);
    StageTimer timer(WPCD_STAGE_FILL_SWAVE, st);
#define WPCD_LAUNCH_SW(L, Q) fill_swave_kernel<L, Q><<<blocks, 256, 0, st>>>(qr, g->p_dev, g->q_dev, g->n_q, n_quad, ch->g0, nnz_geo, \
                                                                            ws.geo_col, ws.geo_row, ws.geo_phi, col_idx, values)
    if (rule == 2) {
        lpe = 8; threads = nnz_geo * lpe; blocks = (int)((threads + 255) / 256);
        fill_swave_analytic_kernel<8><<<blocks, 256, 0, st>>>(qr, g->p_dev, g->q_dev, g->n_q, n_quad, ch->g0, nnz_geo, ws.geo_col, ws.geo_row,
                                                              ws.geo_phi, col_idx, values);
        ++g_launches;
        return cudaGetLastError();
    }
    if (rule == 1) {
        // the rule has up to 3 n work items per element: eight lanes each
        lpe = 8; threads = nnz_geo * lpe; blocks = (int)((threads + 255) / 256);
        if (n_quad == 8) fill_swave_split_kernel<8, 8><<<blocks, 256, 0, st>>>(qr, g->p_dev, g->q_dev, g->n_q, n_quad, ch->g0, nnz_geo, ws.geo_col,
                                                                                ws.geo_row, ws.geo_phi, col_idx, values);
        else fill_swave_split_kernel<8, 0><<<blocks, 256, 0, st>>>(qr, g->p_dev, g->q_dev, g->n_q, n_quad, ch->g0, nnz_geo, ws.geo_col,
                                                                    ws.geo_row, ws.geo_phi, col_idx, values);
        ++g_launches;
        return cudaGetLastError();
    }
    // order 8: two lanes per element once there are enough elements to fill the chip (the per-element
    // prologue -- cell loads, normalisation -- is then paid twice instead of eight times), eight lanes otherwise
    if (n_quad == 8 && nnz_geo >= 65536) { lpe = 2; threads = nnz_geo * lpe; blocks = (int)((threads + 255) / 256); WPCD_LAUNCH_SW(2, 8); }
    else if (n_quad == 8) WPCD_LAUNCH_SW(8, 8);
    else if (n_quad == 10) WPCD_LAUNCH_SW(2, 10);
    else switch (lpe) {
    case 8: WPCD_LAUNCH_SW(8, 0); break;
    case 4: WPCD_LAUNCH_SW(4, 0); break;
    case 2: WPCD_LAUNCH_SW(2, 0); break;
    default: WPCD_LAUNCH_SW(1, 0); break;
    }
#undef WPCD_LAUNCH_SW
    ++g_launches;
    return cudaGetLastError();
}

}  // namespace wpcd_detail
