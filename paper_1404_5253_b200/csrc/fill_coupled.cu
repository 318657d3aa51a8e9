// fill_coupled.cu -- paper step 3 for coupled channels (configs 3-5):
// value[gamma,gamma'] = norm * sum_{k,l1,l1'} g * integral of F P_k(x) cos^{A+1} sin^{B+1} /
// (zeta1^{l'+1} zeta2^{l+1}) over (phi, x), (A15) with reading R1 (A = l1+l1',
// B = l+l'-A).  The geometry (F, zeta, limits) is shared by ALL channel pairs of a geometric
// element, so the work is split in two kernels:
//
//   moments kernels  one warp per geometric element.  With the x-sum factored out,
//                      M[k,A,l,l'] = sum_m  W_m c_m^{A+1} s_m^{B+1}  I_m[k,l,l'],
//                      I_m[k,l,l'] = sum_r  P_k(x_r) T_r[l,l'],   T_r[l,l'] = w_r F_r zeta1^{-(l'+1)} zeta2^{-(l+1)}.
//                    lanes = phi-nodes for the phi set-up, = (phi-node, x-node) pairs for the node set-up;
//                    I_m = P^T T, a small dense contraction (K1 x n)(n x n_ll), runs on the FP64 tensor cores
//                    (mma.sync m8n8k4, SASS DMMA); lanes = monomials for the final multiply-add with the c^a s^b
//                    table.  moments2_kernel: the production path (plain rule, 5 <= n <= 12; transposed conflict-free
//                    tables, power tables instead of T); moments_kernel: kink-split rule and every other order.
//                    Moments are written element-major, moments[element][mu].
//   contract_kernel  value[element][pair] = sum_m M[element][m] G[pair][m] on the FP64 tensor cores, pairs grouped by
//                    (l, l') and by monomial set (wpcd_internal.h); persistent CTAs pull (group, tile block) units,
//                    keep the group's tables and the block's moments in shared memory and write, per pair, coalesced
//                    runs of CSR values and column indices.
#include <math.h>

#include <mutex>
#include <stdlib.h>

#include <algorithm>

#include "quad_device.cuh"
#include "wpcd_internal.h"

using namespace wpcd_quad;
using wpcd_detail::QuadRule;

namespace {

constexpr int MOM_MAX_WARPS = 1;  // warps (= elements) per CTA.  One warp with __launch_bounds__(32) beats two with (64) on config 3
                                  // (1.48 -> 1.29 ms: the compiler schedules with more registers), costs 0-4 % on the moments of
                                  // configs 4-5 (0.5 % of their step); one warp under __launch_bounds__(64) gains nothing; four lose
constexpr int NODE_F = 10;   // doubles per staged phi-node

struct MomentShape {
    int n;        // quadrature order
    int NS;       // phi-node slots staged per warp: n, or max(n, 28) for the kink-split rule (7 u-pieces x 4 items)
    int G;        // phi-nodes handled together by the node set-up
    int K1;       // k_max + 1
    int SP;       // row stride of the P_k table:  8 ceil(K1 / 8) + 4   (conflict-free fragment loads)
    int ST;       // row stride of the T table:    8 ceil(n_ll / 8) + 4
    int IS;       // row stride of the I table:    8 ceil(n_ll / 8) + 2
    int LM1;      // l_max + 1
    int CP;       // 2 l_max + 3 powers of cos / sin
    int n_ab;     // distinct (A+1, B+1) exponent pairs
    int n_ll, n_trip, n_mu;
};

__host__ __device__ inline int moment_smem_doubles(const MomentShape& s)
{
    const int rows = s.G * s.n;
    return (s.NS * NODE_F + rows * (s.SP + s.ST) + s.K1 * s.IS + s.G * 2 * s.CP + s.n_ab + 1) & ~1;   // even: 16-byte pieces
}

// D (8x8) += A (8x4, row) * B (4x8, col), FP64 tensor-core MMA.  Fragment layout: a = A[lane/4][lane%4],
// b = B[lane%4][lane/4], (c0, c1) = C[lane/4][2 (lane%4) + {0,1}].
__device__ __forceinline__ void dmma_884(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// I[k][l,l'] = sum_r P_k(x_r) T_r[l,l'] for one phi-node: (K1 x n) (n x n_ll) in 8x8x4 MMAs.
// Pg / Tg point at this lane's fragment element of x-node (lane % 4); rows r >= n read as zero.
template <int KT>
__device__ __forceinline__ void node_mma(const double* __restrict__ Pg, const double* __restrict__ Tg, int n, int K1, int SP, int ST,
                                         int MT, int NT, double* __restrict__ Ib, int IS, int lane)
{
    bool live[KT];
#pragma unroll
    for (int kt = 0; kt < KT; ++kt) live[kt] = kt * 4 + (lane & 3) < n;
    double* Io = Ib + (lane >> 2) * IS + 2 * (lane & 3);
    for (int mt = 0; mt < MT; ++mt) {
        double a[KT];
#pragma unroll
        for (int kt = 0; kt < KT; ++kt) a[kt] = live[kt] ? Pg[kt * 4 * SP + mt * 8] : 0.0;
        for (int nt = 0; nt < NT; ++nt) {
            double c0 = 0.0, c1 = 0.0;
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) dmma_884(c0, c1, a[kt], live[kt] ? Tg[kt * 4 * ST + nt * 8] : 0.0);
            if (mt * 8 + (lane >> 2) < K1) *reinterpret_cast<double2*>(Io + mt * 8 * IS + nt * 8) = make_double2(c0, c1);
        }
    }
}

__device__ __forceinline__ double ipow_small(double b, int e)   // e < 64
{
    double r = 1.0;
#pragma unroll
    for (int bit = 0; bit < 6; ++bit) { if (e & (1 << bit)) r *= b; b *= b; }
    return r;
}

// Moment layout: element-major, moments[element - e_begin][mu] (coalesced stores here; the contraction stages the
// contiguous range of one l-group per element).
template <int MAXS, bool SPLIT>
__global__ void __launch_bounds__(MOM_MAX_WARPS * 32, 16)
moments_kernel(const __grid_constant__ QuadRule rule, const double* __restrict__ p, const double* __restrict__ q, int n_q, MomentShape sh,
               int64_t e_begin, int64_t e_end, const int32_t* __restrict__ geo_col, const int32_t* __restrict__ geo_row,
               const double2* __restrict__ geo_phi, const int32_t* __restrict__ ll_pack, const int32_t* __restrict__ trip_pack,
               const int32_t* __restrict__ mu_pack, const int32_t* __restrict__ ab_pack, double* __restrict__ moments)
{
    extern __shared__ double sm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = sh.n, G = sh.G, K1 = sh.K1, SP = sh.SP, ST = sh.ST, IS = sh.IS, LM1 = sh.LM1, CP = sh.CP, n_ab = sh.n_ab;
    const int n_ll = sh.n_ll, n_trip = sh.n_trip, n_mu = sh.n_mu;
    // block-shared tables: ll_of[(l, l')] -> ll index (or -1), trip_pack
    int32_t* ll_of = reinterpret_cast<int32_t*>(sm);                     // [LM1*LM1]
    int32_t* trip_s = ll_of + LM1 * LM1;                                  // [n_trip]
    double* wbase = sm + ((((LM1 * LM1 + n_trip + 1) >> 1) + 1) & ~1);
    for (int t = threadIdx.x; t < LM1 * LM1; t += blockDim.x) ll_of[t] = -1;
    __syncthreads();
    for (int t = threadIdx.x; t < n_ll; t += blockDim.x) { const int v = ll_pack[t]; ll_of[(v & 0xff) * LM1 + (v >> 8)] = t; }
    for (int t = threadIdx.x; t < n_trip; t += blockDim.x) trip_s[t] = trip_pack[t];
    __syncthreads();
    const int64_t e = e_begin + (int64_t)blockIdx.x * (blockDim.x >> 5) + warp;
    if (e >= e_end) return;
    const bool full_ll = n_ll == LM1 * LM1;                           // every (l, l') present: ll = l * LM1 + l'
    double* nodeS = wbase + (size_t)warp * moment_smem_doubles(sh);   // [NS][NODE_F]
    double* Pk = nodeS + sh.NS * NODE_F;                                  // [G*n][SP]    P_k(x_r)
    double* T = Pk + G * n * SP;                                      // [G*n][ST]    T_r[l,l']
    double* Ib = T + G * n * ST;                                      // [K1][IS]     I[k][l,l'] of one phi-node
    double* cs = Ib + K1 * IS;                                        // [G][2][CP]   powers of cos, sin
    double* csp = cs + G * 2 * CP;                                    // [n_ab]       c^a s^b of one phi-node

    // per monomial: offset into Ib (low 16 bits) and into csp (high 16 bits)
    int pk[MAXS];
    double acc[MAXS];
#pragma unroll
    for (int s = 0; s < MAXS; ++s) {
        const int m = lane + 32 * s;
        acc[s] = 0.0;
        pk[s] = -1;
        if (m < n_mu) {
            const int v = mu_pack[m], tp = trip_s[v & 0xffff];
            pk[s] = ((tp & 0xff) * IS + (tp >> 8)) | ((v >> 16) << 16);     // mu_pack: triple | ab index << 16
        }
    }
    const int col = geo_col[e], row = geo_row[e];
    const double2 ph = geo_phi[e];
    const Cell z = load_cell(p, q, n_q, row, col);
    const CellSq zs = square_cell(z);
    const double norm = cell_norm(z);
    const double half_phi = 0.5 * (ph.y - ph.x), mid_phi = 0.5 * (ph.x + ph.y);
    const int MT = (SP - 4) >> 3, NT = (ST - 4) >> 3, KT = (n + 3) >> 2;
    // steps 2-4 for the V phi-node slots staged in nodeS (slot: weight in phi (0 = skip), C, S, Lq^2, Uq^2, b1, b2, beta,
    // and the u-interval the inner rule runs on)
    auto process = [&](const int V) {
        for (int m0 = 0; m0 < V; m0 += G) {
            const int cnt = min(G, V - m0);
            // ---- step 2: node set-up, lane = (phi-node g, x-node r)
            for (int idx = lane; idx < cnt * n; idx += 32) {
                const int g = idx / n, r = idx - g * n;
                const double* o = nodeS + (m0 + g) * NODE_F;
                if (o[0] == 0.0) continue;
                PhiNodeSq s;
                s.Lq2 = o[3]; s.Uq2 = o[4];
                const double b1 = o[5], b2 = o[6], beta = o[7], u_lo = o[8], u_hi = o[9];
                const double half_u = 0.5 * (u_hi - u_lo), mid_u = 0.5 * (u_lo + u_hi);
                const double u = mid_u + half_u * rule.xi[r];
                const double x = u - 1.0;
                const double iz1 = rsqrt(b1 + beta * u), iz2 = rsqrt(b2 + beta * u);
                const double wF = (o[0] * norm) * (half_u * rule.w[r]) * 0.5 * twoF_A14_sq(zs, s, iz1 * iz1, iz2 * iz2);
                double* Pr = Pk + (g * n + r) * SP;
                double p0 = 1.0, p1 = x;
                Pr[0] = 1.0;
                if (K1 > 1) Pr[1] = x;
                for (int k = 2; k < K1; ++k) {
                    const double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) * rule.invk[k];
                    Pr[k] = p2;
                    p0 = p1; p1 = p2;
                }
                double* Tr = T + (g * n + r) * ST;
                double z2pow = wF * iz2;                                  // wF zeta2^{-(l+1)}
                if (full_ll) {
                    for (int l = 0; l < LM1; ++l) {
                        double both = z2pow * iz1;                        // ... zeta1^{-(l'+1)}
                        for (int lp = 0; lp < LM1; ++lp) { Tr[l * LM1 + lp] = both; both *= iz1; }
                        z2pow *= iz2;
                    }
                } else {
                    for (int l = 0; l < LM1; ++l) {
                        double both = z2pow * iz1;
                        for (int lp = 0; lp < LM1; ++lp) {
                            const int ll = ll_of[l * LM1 + lp];
                            if (ll >= 0) Tr[ll] = both;
                            both *= iz1;
                        }
                        z2pow *= iz2;
                    }
                }
            }
            for (int idx = lane; idx < cnt * CP; idx += 32) {
                const int g = idx / CP, ex = idx - g * CP;
                const double* o = nodeS + (m0 + g) * NODE_F;
                cs[(g * 2 + 0) * CP + ex] = ipow_small(o[1], ex);
                cs[(g * 2 + 1) * CP + ex] = ipow_small(o[2], ex);
            }
            __syncwarp();
            for (int g = 0; g < cnt; ++g) {
                if (nodeS[(m0 + g) * NODE_F] == 0.0) continue;           // warp-uniform
                // c^a s^b table of this phi-node
                for (int idx = lane; idx < n_ab; idx += 32) {
                    const int ab = ab_pack[idx];
                    csp[idx] = cs[(g * 2 + 0) * CP + (ab & 0xff)] * cs[(g * 2 + 1) * CP + (ab >> 8)];
                }
                // ---- step 3: I[k][l,l'] = sum_r P_k(x_r) T_r[l,l'] on the FP64 tensor cores
                const double* Pg = Pk + (g * n + (lane & 3)) * SP + (lane >> 2);
                const double* Tg = T + (g * n + (lane & 3)) * ST + (lane >> 2);
                switch (KT) {
                case 1: node_mma<1>(Pg, Tg, n, K1, SP, ST, MT, NT, Ib, IS, lane); break;
                case 2: node_mma<2>(Pg, Tg, n, K1, SP, ST, MT, NT, Ib, IS, lane); break;
                case 3: node_mma<3>(Pg, Tg, n, K1, SP, ST, MT, NT, Ib, IS, lane); break;
                case 4: node_mma<4>(Pg, Tg, n, K1, SP, ST, MT, NT, Ib, IS, lane); break;
                default:
                    for (int mt = 0; mt < MT; ++mt)
                        for (int nt = 0; nt < NT; ++nt) {
                            double c0 = 0.0, c1 = 0.0;
                            for (int kt = 0; kt < KT; ++kt) {
                                const bool live = kt * 4 + (lane & 3) < n;
                                dmma_884(c0, c1, live ? Pg[kt * 4 * SP + mt * 8] : 0.0, live ? Tg[kt * 4 * ST + nt * 8] : 0.0);
                            }
                            if (mt * 8 + (lane >> 2) < K1) *reinterpret_cast<double2*>(Ib + (mt * 8 + (lane >> 2)) * IS + nt * 8 + 2 * (lane & 3)) = make_double2(c0, c1);
                        }
                    break;
                }
                __syncwarp();
                // ---- step 4: M[mu] += c^{A+1} s^{B+1} I[k][l,l'], lane = monomial
#pragma unroll
                for (int s = 0; s < MAXS; ++s) {
                    const int v = pk[s];
                    if (v >= 0) acc[s] = fma(csp[v >> 16], Ib[v & 0xffff], acc[s]);
                }
                __syncwarp();
            }
        }
    };
    if (ph.x < ph.y) {
        if (!SPLIT) {
            // ---- step 1: everything that depends on phi only, one lane per phi-node
            for (int m = lane; m < n; m += 32) {
                PhiNodeSq s;
                const bool ok = phi_node_sq(z, zs, mid_phi + half_phi * rule.xi[m], s);
                double* o = nodeS + m * NODE_F;
                o[0] = ok ? half_phi * rule.w[m] : 0.0; o[1] = s.C; o[2] = s.S; o[3] = s.Lq2; o[4] = s.Uq2;
                o[5] = s.b1; o[6] = s.b2; o[7] = s.beta; o[8] = s.u_lo; o[9] = s.u_hi;
            }
            __syncwarp();
            process(n);
        } else {
            // ---- kink-split rule RS(n) (R14): items = (phi-piece, phi-node); an item stages one slot per
            // u-piece (at most 7), IPR items per round so that a round always fits the NS slots
            double pc[SPLIT_MAX_PHI + 1];
            const int n_items = split_phi(z, ph.x, ph.y, pc) * n;
            const int IPR = sh.NS / SPLIT_MAX_U;
            for (int i0 = 0; i0 < n_items; i0 += IPR) {
                const int item = i0 + lane;
                int np = 0;
                PhiNodeSq s;
                double cand[6];
                double wphi = 0.0;
                if (lane < IPR && item < n_items) {
                    const int piece = item / n, m = item - piece * n;
                    const double pa = piece == 0 ? pc[0] : (piece == 1 ? pc[1] : pc[2]);
                    const double pb = piece == 0 ? pc[1] : (piece == 1 ? pc[2] : pc[3]);
                    const double hp = 0.5 * (pb - pa);
                    if (phi_node_sq(z, zs, 0.5 * (pa + pb) + hp * rule.xi[m], s)) {
                        split_u_candidates(z, zs, s, cand);
                        wphi = hp * rule.w[m];
                        double lower = s.u_lo;
                        np = 1;
#pragma unroll
                        for (int i = 0; i < 6; ++i)
                            if (cand[i] > lower && cand[i] < s.u_hi) { ++np; lower = cand[i]; }
                    }
                }
                int off = np;                                    // inclusive scan over the lanes
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int t = __shfl_up_sync(0xffffffffu, off, d);
                    if (lane >= d) off += t;
                }
                const int V = __shfl_sync(0xffffffffu, off, 31);
                off -= np;
                if (np > 0) {
                    double lower = s.u_lo;
                    auto put = [&](double lo, double hi) {
                        double* o = nodeS + off * NODE_F;
                        o[0] = wphi; o[1] = s.C; o[2] = s.S; o[3] = s.Lq2; o[4] = s.Uq2;
                        o[5] = s.b1; o[6] = s.b2; o[7] = s.beta; o[8] = lo; o[9] = hi;
                        ++off;
                    };
#pragma unroll
                    for (int i = 0; i < 6; ++i)
                        if (cand[i] > lower && cand[i] < s.u_hi) { put(lower, cand[i]); lower = cand[i]; }
                    put(lower, s.u_hi);
                }
                __syncwarp();
                process(V);
            }
        }
    }
    double* out = moments + (size_t)(e - e_begin) * n_mu;       // element-major: one contiguous row per element
#pragma unroll
    for (int s = 0; s < MAXS; ++s)
        if (lane + 32 * s < n_mu) out[lane + 32 * s] = acc[s];
}

// ---------------------------------------------------------------------------------------------------------------
// moments2_kernel -- the same moments for the plain rule R(n), 5 <= n <= 12, k_max <= 15: the production path.
// One warp per geometric element.  Differences from moments_kernel (kept for the kink-split rule and the other orders):
//   * the tables are stored TRANSPOSED, [quantity][node slot]: the lanes that set up the nodes write consecutive words,
//     and with a row stride = 4 (mod 16) the MMA fragment loads are conflict-free as well;
//   * T[l,l'] = wF zeta2^{-(l+1)} zeta1^{-(l'+1)} is never stored: two small power tables pa[l] = wF zeta2^{-(l+1)},
//     pb[l'] = zeta1^{-(l'+1)} (2 (l_max+1) values per node instead of (l_max+1)^2) and one multiply when a B fragment
//     is formed; node slots are padded to a multiple of 4 per phi-node with zeros, so no fragment needs a mask;
//   * B fragments are formed once per (n-tile, k-step) and used for every m-tile; the MMAs are free to interleave.
struct MomentShape2 {
    int n;        // quadrature order
    int G;        // phi-nodes whose x-nodes are set up together (G n <= 32 lanes)
    int NP;       // node slots per phi-node: n rounded up to a multiple of 4 (KT = NP / 4 k-steps)
    int RS;       // row stride of the transposed tables: >= G NP, = 4 (mod 16)
    int K1;       // k_max + 1
    int NT;       // n-tiles: ceil(n_ll / 8)
    int IS;       // row stride of the I table: 8 NT + 2
    int LM1;      // l_max + 1
    int CP;       // 2 l_max + 3 powers of cos / sin
    int n_ab, n_ll, n_mu;
};

__host__ __device__ inline int moment2_smem_doubles(const MomentShape2& s)
{
    // phi-node records | P_k [K1][RS] | pa [LM1 + 1][RS] (last row zero) | pb [LM1][RS] | I [K1][IS] | cos/sin powers [G][2][CP] | c^a s^b [n_ab]
    return (s.n * NODE_F + s.K1 * s.RS + (2 * s.LM1 + 1) * s.RS + s.K1 * s.IS + s.G * 2 * s.CP + s.n_ab + 1) & ~1;
}

#ifndef MOM_HOIST_MAX
#define MOM_HOIST_MAX 14
#endif
template <int MAXS, int KT, int MT>
__global__ void __launch_bounds__(32, 16)
moments2_kernel(const __grid_constant__ QuadRule rule, const double* __restrict__ p, const double* __restrict__ q, int n_q, MomentShape2 sh,
                int64_t e_begin, int64_t e_end, const int32_t* __restrict__ geo_col, const int32_t* __restrict__ geo_row,
                const double2* __restrict__ geo_phi, const int32_t* __restrict__ ll_pack, const int32_t* __restrict__ mu_ib_pack,
                const int32_t* __restrict__ ab_pack, double* __restrict__ moments)
{
    extern __shared__ double sm[];
    const int lane = threadIdx.x, quad = lane & 3, oct = lane >> 2;
    const int n = sh.n, G = sh.G, NP = sh.NP, RS = sh.RS, K1 = sh.K1, NT = sh.NT, IS = sh.IS, LM1 = sh.LM1, CP = sh.CP, n_ab = sh.n_ab;
    const int n_ll = sh.n_ll, n_mu = sh.n_mu;
    const int64_t e = e_begin + blockIdx.x;
    if (e >= e_end) return;
    double* nodeS = sm;                       // [n][NODE_F]
    double* Pt = nodeS + n * NODE_F;          // [K1][RS]   P_k(x) of node slot g NP + r
    double* pa = Pt + K1 * RS;                // [LM1 + 1][RS]  wF zeta2^{-(l+1)}; row LM1 stays zero (columns beyond n_ll)
    double* pb = pa + (LM1 + 1) * RS;         // [LM1][RS]  zeta1^{-(l'+1)}
    double* Ib = pb + LM1 * RS;               // [K1][IS]   I[k][l,l'] of one phi-node
    double* cs = Ib + K1 * IS;                // [G][2][CP] powers of cos, sin
    double* csp = cs + G * 2 * CP;            // [n_ab]     c^a s^b of one phi-node
    // the padding slots of the power tables must read as zero (they feed the MMAs); P_k only has to be finite there
    for (int i = lane; i < (K1 + 2 * LM1 + 1) * RS; i += 32) Pt[i] = 0.0;
    // per monomial: BYTE offsets from sm of its I entry (low 16 bits) and of its c^a s^b entry (high 16 bits): the multiply-add
    // of step 4 then needs no address arithmetic beyond one mask / shift, and no predicate -- a slot beyond n_mu points both
    // at a word of the zero row of pa (the whole block of a warp is < 64 KB, checked by the host)
    const unsigned off_zero = (unsigned)((pa + LM1 * RS - sm) * sizeof(double));
    const unsigned off_ib = (unsigned)((Ib - sm) * sizeof(double)), off_csp = (unsigned)((csp - sm) * sizeof(double));
    unsigned pk[MAXS];
    double acc[MAXS];
#pragma unroll
    for (int s = 0; s < MAXS; ++s) {
        const int m = lane + 32 * s;
        acc[s] = 0.0;
        pk[s] = (off_zero << 16) | off_zero;
        if (m < n_mu) {
            const unsigned v = (unsigned)mu_ib_pack[m];                       // (k IS + ll) | ab index << 16
            pk[s] = ((off_csp + 8u * (v >> 16)) << 16) | (off_ib + 8u * (v & 0xffffu));
        }
    }
    const char* smb = reinterpret_cast<const char*>(sm);
    // this lane's (up to two) entries of the c^a s^b table: byte offsets of c^a and s^b inside a phi-node's power block
    unsigned abo[2];
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int idx = lane + 32 * j;
        const int ab = idx < n_ab ? ab_pack[idx] : 0;
        abo[j] = (8u * (unsigned)(ab & 0xff) << 16) | 8u * (unsigned)(CP + (ab >> 8));
    }
    // this lane's (l, l') of every n-tile: where its rows of the power tables start (a column beyond n_ll reads the zero row)
    const double* qa[4];
    const double* qb[4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
        const int ll = nt * 8 + oct;
        qa[nt] = pa + LM1 * RS + quad; qb[nt] = pb + quad;
        if (nt < NT && ll < n_ll) { const int v = ll_pack[ll]; qa[nt] = pa + (v & 0xff) * RS + quad; qb[nt] = pb + (v >> 8) * RS + quad; }
    }
    const double* qp[MT];          // this lane's rows of the P table (a row beyond K1 reads the zero row of pa)
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) qp[mt] = mt * 8 + oct < K1 ? Pt + (mt * 8 + oct) * RS + quad : pa + LM1 * RS + quad;
    const int col = geo_col[e], row = geo_row[e];
    const double2 ph = geo_phi[e];
    const Cell z = load_cell(p, q, n_q, row, col);
    const CellSq zs = square_cell(z);
    const double norm = cell_norm(z);
    const double half_phi = 0.5 * (ph.y - ph.x), mid_phi = 0.5 * (ph.x + ph.y);
    __syncwarp();
    if (ph.x < ph.y) {
        // ---- step 1: everything that depends on phi only, one lane per phi-node (weight 0: the node contributes nothing)
        for (int m = lane; m < n; m += 32) {
            PhiNodeSq s;
            const bool ok = phi_node_sq(z, zs, mid_phi + half_phi * rule.xi[m], s);
            double* o = nodeS + m * NODE_F;
            o[0] = ok ? half_phi * rule.w[m] : 0.0; o[1] = s.C; o[2] = s.S; o[3] = s.Lq2; o[4] = s.Uq2;
            o[5] = s.b1; o[6] = s.b2; o[7] = s.beta; o[8] = s.u_lo; o[9] = s.u_hi;
        }
        __syncwarp();
        for (int m0 = 0; m0 < n; m0 += G) {
            const int cnt = min(G, n - m0);
            // ---- step 2: node set-up, lane = (phi-node g, x-node r) -> slot g NP + r of the transposed tables
            if (lane < cnt * n) {
                const int g = lane / n, r = lane - g * n, slot = g * NP + r;
                const double* o = nodeS + (m0 + g) * NODE_F;
                if (o[0] != 0.0) {
                    PhiNodeSq s;
                    s.Lq2 = o[3]; s.Uq2 = o[4];
                    const double b1 = o[5], b2 = o[6], beta = o[7], u_lo = o[8], u_hi = o[9];
                    const double half_u = 0.5 * (u_hi - u_lo), mid_u = 0.5 * (u_lo + u_hi);
                    const double u = mid_u + half_u * rule.xi[r];
                    const double x = u - 1.0;
                    const double iz1 = rsqrt(b1 + beta * u), iz2 = rsqrt(b2 + beta * u);
                    const double wF = (o[0] * norm) * (half_u * rule.w[r]) * 0.5 * twoF_A14_sq(zs, s, iz1 * iz1, iz2 * iz2);
                    double p0 = 1.0, p1 = x;
                    Pt[slot] = 1.0;
                    if (K1 > 1) Pt[RS + slot] = x;
                    for (int k = 2; k < K1; ++k) {
                        const double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) * rule.invk[k];
                        Pt[k * RS + slot] = p2;
                        p0 = p1; p1 = p2;
                    }
                    double za = wF * iz2, zb = iz1;                   // wF zeta2^{-(l+1)}, zeta1^{-(l'+1)}
                    for (int l = 0; l < LM1; ++l) {
                        pa[l * RS + slot] = za; pb[l * RS + slot] = zb;
                        za *= iz2; zb *= iz1;
                    }
                }
            }
            // powers of cos, sin of the group's phi-nodes: lane = (phi-node, cos | sin), running product
            if (lane < 2 * cnt) {
                const double base = nodeS[(m0 + (lane >> 1)) * NODE_F + 1 + (lane & 1)];
                double* d = cs + lane * CP;
                double pw = 1.0;
                for (int ex = 0; ex < CP; ++ex) { d[ex] = pw; pw *= base; }
            }
            __syncwarp();
            for (int g = 0; g < cnt; ++g) {
                if (nodeS[(m0 + g) * NODE_F] == 0.0) continue;           // warp-uniform
                // c^a s^b table of this phi-node
                {
                    const char* csg = reinterpret_cast<const char*>(cs + g * 2 * CP);
#pragma unroll
                    for (int j = 0; j < 2; ++j)
                        if (lane + 32 * j < n_ab)
                            csp[lane + 32 * j] = *reinterpret_cast<const double*>(csg + (abo[j] >> 16)) * *reinterpret_cast<const double*>(csg + (abo[j] & 0xffffu));
                    for (int idx = lane + 64; idx < n_ab; idx += 32) {      // more than 64 exponent pairs: not for l <= 4
                        const int ab = ab_pack[idx];
                        csp[idx] = cs[(g * 2 + 0) * CP + (ab & 0xff)] * cs[(g * 2 + 1) * CP + (ab >> 8)];
                    }
                }
                // ---- step 3: I[k][l,l'] = sum_r P_k(x_r) T_r[l,l'] on the FP64 tensor cores
                const int s0 = g * NP;                                 // first node slot of this phi-node
                double a[MT][KT];
#pragma unroll
                for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                    for (int kt = 0; kt < KT; ++kt) a[mt][kt] = qp[mt][s0 + 4 * kt];
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                    if (nt >= NT) break;
                    double b[KT];
#pragma unroll
                    for (int kt = 0; kt < KT; ++kt) b[kt] = qa[nt][s0 + 4 * kt] * qb[nt][s0 + 4 * kt];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        double c0 = 0.0, c1 = 0.0;
#pragma unroll
                        for (int kt = 0; kt < KT; ++kt) dmma_884(c0, c1, a[mt][kt], b[kt]);
                        if (mt * 8 + oct < K1) *reinterpret_cast<double2*>(Ib + (mt * 8 + oct) * IS + nt * 8 + 2 * quad) = make_double2(c0, c1);
                    }
                }
                __syncwarp();
                // ---- step 4: M[mu] += c^{A+1} s^{B+1} I[k][l,l'], lane = monomial
#pragma unroll
                for (int s = 0; s < MAXS; ++s) {
                    unsigned v = pk[s];
                    if (MAXS > MOM_HOIST_MAX) asm volatile("" : "+r"(v));      // many slots: the two addresses are formed here, not kept in registers
                    acc[s] = fma(*reinterpret_cast<const double*>(smb + (v >> 16)), *reinterpret_cast<const double*>(smb + (v & 0xffffu)), acc[s]);
                }
                __syncwarp();
            }
        }
    }
    double* out = moments + (size_t)(e - e_begin) * n_mu;       // element-major: one contiguous row per element
#pragma unroll
    for (int s = 0; s < MAXS; ++s)
        if (lane + 32 * s < n_mu) out[lane + 32 * s] = acc[s];
}

}  // namespace

namespace {

constexpr int CT_THREADS = 256;
constexpr int CT_WARPS = CT_THREADS / 32;
constexpr int CT_E = WPCD_CT_ELEMS;
constexpr int CT_MAX_TILES = 8;          // 32-element tiles per work unit, at most

// (grp, cnt, gcol, row) of every geometric element: what the contraction needs to place its values.
__global__ void __launch_bounds__(256)
elem_rec_kernel(int64_t nnz_geo, const int32_t* __restrict__ geo_col, const int32_t* __restrict__ geo_row,
                const int32_t* __restrict__ geo_row_ptr, int4* __restrict__ rec)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nnz_geo) return;
    const int r = geo_row[e], grp = geo_row_ptr[r];
    rec[e] = make_int4(grp, geo_row_ptr[r + 1] - grp, geo_col[e], r);
}

// The same MMA without "volatile": the compiler may interleave independent accumulator chains.
__device__ __forceinline__ void dmma_884_nv(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Contraction.  Work unit = ((l, l') group, block of n_tb tiles of 32 consecutive geometric elements).
// The CTA copies the group's tables (items, pair records, monomial positions, coefficient fragments: one blob) to shared
// memory, stages the block's moments of that (l, l') range (element-major rows,
// one contiguous piece per element) and deals (item, tile) pieces to its warps, no barrier in between.  Piece:
// D[element][pair] = M[element][monomial] G[pair][monomial] on the FP64 tensor cores, every operand from shared memory;
// then the 8 x 32 results go through a small per-warp buffer so that lane = element: a pair's values for the elements of
// one geometric row are consecutive in CSR row (gamma, r), and a warp store covers the tile's piece of that row (the
// neighbouring tile, handled by the same CTA in the same unit or within microseconds, continues it).
__global__ void __launch_bounds__(CT_THREADS, 3)
contract_kernel(int64_t e0, int64_t e1, int64_t nnz_geo, int n_geo, const int4* __restrict__ elem_rec, unsigned int* __restrict__ ticket,
                const double* __restrict__ moments, int n_mu, const wpcd_ct_group* __restrict__ groups, int n_groups,
                const unsigned char* __restrict__ blob, int tab_bytes, int n_tb, int ms_stride, int32_t* __restrict__ col_idx,
                double* __restrict__ values)
{
    extern __shared__ __align__(16) unsigned char ct_sm[];
    unsigned char* tab = ct_sm;                                                         // the group's blob
    double* Ms = reinterpret_cast<double*>(ct_sm + tab_bytes);                          // [n_tb * 32][ms_stride]
    double* Sw = Ms + (size_t)n_tb * CT_E * ms_stride + (threadIdx.x >> 5) * (8 * 33);  // this warp's [8][33] transposition buffer
    int4* rec_s = reinterpret_cast<int4*>(Ms + (size_t)n_tb * CT_E * ms_stride + CT_WARPS * 8 * 33);   // [n_tb * 32]
    __shared__ longlong2 Pw_all[CT_WARPS][8];      // per warp: the current item's pairs, (row-block start, ncoupled << 32 | rank)
    __shared__ int Gw_all[CT_WARPS][8];            //                                      gamma' * n_geo
    longlong2* Pw = Pw_all[threadIdx.x >> 5];
    int* Gw = Gw_all[threadIdx.x >> 5];
    __shared__ unsigned int s_unit;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, quad = lane & 3, oct = lane >> 2;
    const int64_t n_tiles = (e1 - e0 + CT_E - 1) / CT_E;
    const int64_t n_blocks = (n_tiles + n_tb - 1) / n_tb;
    const uint64_t n_units = (uint64_t)n_blocks * n_groups;
    int cur_group = -1;
    wpcd_ct_group g = {0, 0, 0, 0, 0, 0, 0, 0};
    unsigned int next_u = 0;                   // thread 0: the ticket drawn one unit ahead (its round trip hides behind the work)
    if (tid == 0) next_u = atomicAdd(ticket, 1u);
    for (;;) {
        if (tid == 0) s_unit = next_u;
        __syncthreads();                       // also: every warp is done with the previous unit's shared memory
        const unsigned int u = s_unit;
        if (u >= n_units) return;
        if (tid == 0) next_u = atomicAdd(ticket, 1u);
        // tile block after tile block: all values of a block's elements are written within a short time (the pieces of a CSR
        // row written by different groups then meet in L2 before they are evicted)
        const int64_t blk = u / (unsigned)n_groups;
        const int gi = (int)(u - (uint64_t)blk * n_groups);
        if (gi != cur_group) {                 // new group: its tables go to shared memory
            g = groups[gi];
            cur_group = gi;
            const uint4* src = reinterpret_cast<const uint4*>(blob + g.blob_off);
            uint4* dst = reinterpret_cast<uint4*>(tab);
            for (int i = tid; i < (g.blob_bytes >> 4); i += CT_THREADS)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst + i)), "l"(src + i) : "memory");
        }
        const int64_t es = e0 + blk * n_tb * CT_E;
        const int rows = (int)min((int64_t)n_tb * CT_E, e1 - es);
        // ---- stage the moments of this (l, l') for the block's elements: warp = element row, lanes along the monomials
        {
            const double* src = moments + (size_t)(es - e0) * n_mu + g.mu_lo;
            // asynchronous copies (8 bytes each: a row starts on an 8-byte boundary only), all in flight together; the
            // addresses advance by constant strides (an element row is n_mu doubles away from the next)
            const double* s = src + (size_t)warp * n_mu + lane;
            uint32_t d = (uint32_t)__cvta_generic_to_shared(Ms + warp * ms_stride + lane);
            const size_t s_step = (size_t)CT_WARPS * n_mu;
            const uint32_t d_step = (uint32_t)(CT_WARPS * ms_stride * sizeof(double));
            for (int ei = warp; ei < rows; ei += CT_WARPS, s += s_step, d += d_step)
                for (int mi = lane; mi < g.n_mono; mi += 32)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d + 8 * (mi - lane)), "l"(s + (mi - lane)) : "memory");
            for (int i = tid; i < rows; i += CT_THREADS) rec_s[i] = __ldg(elem_rec + es + i);       // grp, cnt, gcol, row
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
        const wpcd_ct_item* items = reinterpret_cast<const wpcd_ct_item*>(tab);
        const int4* prs = reinterpret_cast<const int4*>(tab + g.pairs_off);
        const int32_t* idx_s = reinterpret_cast<const int32_t*>(tab + g.idx_off);
        const double* g_s = reinterpret_cast<const double*>(tab + g.g_off);
        const int n_t = (rows + CT_E - 1) / CT_E;
        const int n_pieces = g.n_items * n_t;
        int ii = warp / n_t, t = warp - ii * n_t;               // piece = (item ii, tile t), item-major, dealt round-robin to the warps
        for (int pc = warp; pc < n_pieces; pc += CT_WARPS) {
            const wpcd_ct_item it = items[ii];
            const int kt = it.kt, np = it.n_pairs;
            // lane q < np: (prefix of ncoupled over gamma, ncoupled(gamma), rank of gamma', gamma') of pair q -> where the pair's
            // values start in the CSR (entry 0 of row (gamma, 0) + rank * 0), its row-block factor, rank and column offset
            if (lane < np) {
                const int4 pr = prs[it.pair_off + lane];
                Pw[lane] = make_longlong2((long long)pr.x * nnz_geo, ((long long)(unsigned)pr.y << 32) | (unsigned)pr.z);
                Gw[lane] = pr.w * n_geo;
            }
            const int ib = it.idx_off + quad, gb = it.g_off + lane;     // [k][np][4]: lane (oct, quad) reads entry oct * 4 + quad = lane of step k
            const bool bl = oct < np;
            const int gstep = 4 * np;
            const int m = min(CT_E, rows - t * CT_E);
            const int o0 = (t * CT_E + min(oct, m - 1)) * ms_stride, o1 = (t * CT_E + min(8 + oct, m - 1)) * ms_stride;
            const int o2 = (t * CT_E + min(16 + oct, m - 1)) * ms_stride, o3 = (t * CT_E + min(24 + oct, m - 1)) * ms_stride;
            double c[4][2];
#pragma unroll
            for (int j = 0; j < 4; ++j) c[j][0] = c[j][1] = 0.0;
#pragma unroll 2
            for (int k = 0; k < kt; ++k) {
                const int mi = idx_s[ib + 4 * k];
                const double b = bl ? g_s[gb + gstep * k] : 0.0;
                dmma_884_nv(c[0][0], c[0][1], Ms[o0 + mi], b);
                dmma_884_nv(c[1][0], c[1][1], Ms[o1 + mi], b);
                dmma_884_nv(c[2][0], c[2][1], Ms[o2 + mi], b);
                dmma_884_nv(c[3][0], c[3][1], Ms[o3 + mi], b);
            }
            // lane holds out[element 8 j + oct][pair 2 quad + h]: transpose through the warp's buffer, row = pair, lane = element
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int j = 0; j < 4; ++j) Sw[(2 * quad + h) * 33 + 8 * j + oct] = c[j][h];
            __syncwarp();
            if (lane < m) {
                const int4 rec = rec_s[t * CT_E + lane];            // this lane's element: grp, cnt, gcol, row
                const int pos = (int)(es - rec.x) + t * CT_E + lane;
                for (int q = 0; q < np; ++q) {
                    const longlong2 pq = Pw[q];                     // (start of the pair's row block, ncoupled << 32 | rank)
                    const int ncoup = (int)(pq.y >> 32), ci = (int)(unsigned)pq.y;
                    const int64_t o = pq.x + (ncoup * rec.x + ci * rec.y + pos);       // < 2^31 inside a row block (checked by the host)
                    __stcs(values + o, Sw[q * 33 + lane]);
                    __stcs(col_idx + o, Gw[q] + rec.z);
                }
            }
            __syncwarp();
            t += CT_WARPS;
            while (t >= n_t) { t -= n_t; ++ii; }
        }
    }
}

}  // namespace

namespace wpcd_detail {

cudaError_t launch_fill_coupled(const wpcd_grid* g, const wpcd_channels* ch, int n_quad, bool split, const QuadRule& qr,
                                int64_t nnz_geo, const Workspace& ws, const int64_t* /*row_ptr*/, const int32_t* geo_row_ptr,
                                int32_t* col_idx, double* values, cudaStream_t st)
{
    cudaError_t err = cudaSuccess;
    if (nnz_geo == 0 || ch->n_pairs == 0) return cudaSuccess;
    if (ch->n_mu > 32 * 32 || 2 * ch->l_max + 2 > 127) return cudaErrorInvalidValue;
    MomentShape sh;
    sh.n = n_quad; sh.NS = split ? std::max(n_quad, 4 * SPLIT_MAX_U) : n_quad;
    sh.G = std::max(1, std::min(32 / n_quad, n_quad <= 8 ? 4 : 2));   // measured: n = 8: 4 beats 2 by 13 %, n = 10: 3 loses to 2
    sh.K1 = ch->k_max + 1; sh.SP = 8 * ((sh.K1 + 7) / 8) + 4;
    sh.ST = 8 * ((ch->n_ll + 7) / 8) + 4; sh.IS = 8 * ((ch->n_ll + 7) / 8) + 2;
    sh.LM1 = ch->l_max + 1; sh.CP = 2 * ch->l_max + 3; sh.n_ab = ch->n_ab;
    sh.n_ll = ch->n_ll; sh.n_trip = ch->n_trip; sh.n_mu = ch->n_mu;
    if ((sh.SP - 4) * sh.IS >= 65536) return cudaErrorInvalidValue;
    const int mom_warps = MOM_MAX_WARPS;
    const size_t mom_smem = sizeof(double) * ((size_t)((((sh.LM1 * sh.LM1 + sh.n_trip + 1) >> 1) + 1) & ~1) + (size_t)mom_warps * moment_smem_doubles(sh));
    if (mom_smem > 227 * 1024) return cudaErrorInvalidValue;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // contraction: the largest group blob + staged moments [n_tb * 32][ms_stride] + one [8][33] transposition buffer per warp
    // + the block's element records.  n_tb: as many tiles per unit as leave room for three CTAs per SM (at least one).
    const int ms_stride = ch->ct_nmono_max | 1;                 // odd: the A-fragment rows of a quarter-warp fall into different banks
    const int tab_bytes = (ch->ct_blob_max + 15) & ~15;
    auto ct_bytes = [&](int n_tb) {
        return (size_t)tab_bytes + sizeof(double) * ((size_t)n_tb * CT_E * ms_stride + (size_t)CT_WARPS * 8 * 33) + sizeof(int4) * (size_t)n_tb * CT_E;
    };
    int n_tb = CT_MAX_TILES;
    while (n_tb > 1 && ct_bytes(n_tb) > (size_t)70 * 1024) --n_tb;
    const size_t ct_smem = ct_bytes(n_tb);
    if (ct_smem > 227 * 1024) return cudaErrorInvalidValue;
    // the contraction places a value with a 32-bit offset inside the row block of its channel
    if ((int64_t)ch->ct_ncoup_max * nnz_geo + nnz_geo >= (int64_t)INT32_MAX) return cudaErrorInvalidValue;
    const int n_geo = g->n_p * g->n_q;
    const int maxs = (ch->n_mu + 31) / 32;
    // the production path (plain rule, 5 <= n <= 12, k_max <= 15, l_max <= 4, <= 640 monomials): moments2_kernel
    MomentShape2 s2;
    s2.n = n_quad; s2.G = std::max(1, std::min(32 / std::max(n_quad, 1), 4)); s2.NP = 4 * ((n_quad + 3) / 4);
    s2.RS = s2.G * s2.NP; while (s2.RS % 16 != 4) ++s2.RS;
    s2.K1 = ch->k_max + 1; s2.NT = (ch->n_ll + 7) / 8; s2.IS = 8 * s2.NT + 2; s2.LM1 = ch->l_max + 1; s2.CP = 2 * ch->l_max + 3;
    s2.n_ab = ch->n_ab; s2.n_ll = ch->n_ll; s2.n_mu = ch->n_mu;
    const bool fast = !split && n_quad >= 5 && n_quad <= 12 && s2.K1 <= 16 && s2.NT <= 4 && maxs <= 20 &&
                      sizeof(double) * (size_t)moment2_smem_doubles(s2) < 65536;     // 16-bit byte offsets inside a warp's block
    const size_t mom2_smem = sizeof(double) * (size_t)moment2_smem_doubles(s2);
#define WPCD_MOM2(MS, SPL)                                                                                                        \
    do {                                                                                                                      \
        err = raise_dyn_smem(moments_kernel<MS, SPL>, mom_smem);           \
        if (err != cudaSuccess) return err;                                                                                   \
        moments_kernel<MS, SPL><<<blocks, mom_warps * 32, mom_smem, st>>>(qr, g->p_dev, g->q_dev, g->n_q, sh, e0, e1, ws.geo_col,      \
                                                                     ws.geo_row, ws.geo_phi, ch->ll_pack_dev,                 \
                                                                     ch->trip_pack_dev, ch->mu_pack_dev, ch->ab_pack_dev, ws.moments);         \
    } while (0)
#define WPCD_MOM(MS) do { if (split) WPCD_MOM2(MS, true); else WPCD_MOM2(MS, false); } while (0)
#define WPCD_MOMF3(MS, KTV, MTV)                                                                                                    \
    do {                                                                                                                          \
        err = raise_dyn_smem(moments2_kernel<MS, KTV, MTV>, mom2_smem);      \
        if (err != cudaSuccess) return err;                                                                                       \
        moments2_kernel<MS, KTV, MTV><<<(unsigned)(e1 - e0), 32, mom2_smem, st>>>(qr, g->p_dev, g->q_dev, g->n_q, s2, e0, e1, ws.geo_col, \
                                                                                  ws.geo_row, ws.geo_phi, ch->ll_pack_dev, ch->mu_ib_pack_dev, \
                                                                                  ch->ab_pack_dev, ws.moments);   \
    } while (0)
#define WPCD_MOMF2(MS, KTV) do { if (s2.K1 <= 8) WPCD_MOMF3(MS, KTV, 1); else WPCD_MOMF3(MS, KTV, 2); } while (0)
#define WPCD_MOMF(MS) do { if (s2.NP == 8) WPCD_MOMF2(MS, 2); else WPCD_MOMF2(MS, 3); } while (0)
    err = raise_dyn_smem(contract_kernel, ct_smem);
    if (err != cudaSuccess) return err;
    {
        StageTimer timer(WPCD_STAGE_GEO_INDEX, st);
        err = cudaMemsetAsync(ws.counters, 0, sizeof(unsigned int) * (size_t)ws.n_chunks, st);
        if (err != cudaSuccess) return err;
        elem_rec_kernel<<<(unsigned)((nnz_geo + 255) / 256), 256, 0, st>>>(nnz_geo, ws.geo_col, ws.geo_row, geo_row_ptr, ws.elem_rec);
        ++g_launches;
        if ((err = cudaGetLastError()) != cudaSuccess) return err;
    }
    int ct_blocks_per_sm = 0;
    err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ct_blocks_per_sm, contract_kernel, CT_THREADS, ct_smem);
    if (err != cudaSuccess) return err;
    const unsigned ct_blocks = (unsigned)(sms * std::max(1, ct_blocks_per_sm));
    int64_t chunk_no = 0;
    for (int64_t e0 = 0; e0 < nnz_geo; e0 += ws.chunk, ++chunk_no) {
        const int64_t e1 = std::min(nnz_geo, e0 + ws.chunk);
        {
            const unsigned blocks = (unsigned)((e1 - e0 + mom_warps - 1) / mom_warps);
            StageTimer timer(WPCD_STAGE_MOMENTS, st);
            if (fast) {            // accumulator slots per lane: ceil(n_mu / 32), in steps of two above 8 (an unused slot still issues)
                if (maxs <= 8) WPCD_MOMF(8);
                else if (maxs <= 10) WPCD_MOMF(10);
                else if (maxs <= 12) WPCD_MOMF(12);
                else if (maxs <= 14) WPCD_MOMF(14);
                else if (maxs <= 16) WPCD_MOMF(16);
                else if (maxs <= 18) WPCD_MOMF(18);
                else WPCD_MOMF(20);
            }
            else if (maxs <= 4) WPCD_MOM(4);
            else if (maxs <= 8) WPCD_MOM(8);
            else if (maxs <= 12) WPCD_MOM(12);
            else if (maxs <= 16) WPCD_MOM(16);
            else if (maxs <= 24) WPCD_MOM(24);
            else WPCD_MOM(32);
            ++g_launches;
            if ((err = cudaGetLastError()) != cudaSuccess) return err;
        }
        {
            StageTimer timer(WPCD_STAGE_CONTRACT, st);
            // persistent CTAs pulling (group, tile block) units from a work queue
            contract_kernel<<<ct_blocks, CT_THREADS, ct_smem, st>>>(e0, e1, nnz_geo, n_geo, ws.elem_rec, ws.counters + chunk_no, ws.moments, ch->n_mu,
                                                                    ch->ct_groups_dev, (int)ch->ct_groups.size(), ch->ct_blob_dev, tab_bytes, n_tb,
                                                                    ms_stride, col_idx, values);
            ++g_launches;
            if ((err = cudaGetLastError()) != cudaSuccess) return err;
        }
    }
#undef WPCD_MOMF
#undef WPCD_MOMF2
#undef WPCD_MOMF3
#undef WPCD_MOM
#undef WPCD_MOM2
    return cudaSuccess;
}

}  // namespace wpcd_detail
