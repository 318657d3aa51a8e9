// fill_coupled.cu -- paper step 3 for coupled channels (configs 3-5):
// value[gamma,gamma'] = norm * sum_{k,l1,l1'} g * integral of F P_k(x) cos^{A+1} sin^{B+1} /
// (zeta1^{l'+1} zeta2^{l+1}) over (phi, x), (A15) with reading R1 (A = l1+l1',
// B = l+l'-A).  The geometry (F, zeta, limits) is shared by ALL channel pairs of a geometric
// element, so the work is split in two kernels:
//
//   moments_kernel   one warp per geometric element.  With the x-sum factored out,
//                      M[k,A,l,l'] = sum_m  W_m c_m^{A+1} s_m^{B+1}  I_m[k,l,l'],
//                      I_m[k,l,l'] = sum_r  P_k(x_r) T_r[l,l'],   T_r[l,l'] = w_r F_r zeta1^{-(l'+1)} zeta2^{-(l+1)}.
//                    lanes = phi-nodes for the phi set-up, = (phi-node, x-node) pairs for the node set-up
//                    that writes P_k and T to shared memory; I_m = P^T T, a small dense contraction
//                    (K1 x n)(n x n_ll), runs on the FP64 tensor cores (mma.sync m8n8k4, SASS DMMA);
//                    lanes = monomials for the final multiply-add with the c^a s^b table.
//                    Moments are written as [tile of 32 elements][mu][32] (256-byte lines per monomial).
//   contract_kernel  value[pair][element] = sum_m G[pair][m] M[m][element] class by class
//                    (wpcd_internal.h): lane = element, the class block of the moment row lives in
//                    REGISTERS, the dense coefficient rows G stream from shared memory as broadcast
//                    128-bit loads.  A CTA owns one slab of classes (copied to shared memory once,
//                    by a TMA bulk copy) and walks over many 32-element tiles, so that the table is
//                    read from L2 a few hundred times in all and every moment exactly once; the next
//                    class block is staged by cp.async while the current one is contracted.  Each
//                    pair writes 32 consecutive CSR values + column indices per warp (coalesced).
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
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
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
__global__ void __launch_bounds__(MOM_MAX_WARPS * 32)
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

}  // namespace

namespace {

constexpr int CT_THREADS = 256;
constexpr int CT_WARPS = CT_THREADS / 32;
constexpr int CT_E = WPCD_CT_ELEMS;

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

// Contraction.  Work unit = (tile of 32 consecutive geometric elements, l-group).  The CTA stages the tile's moments of
// that l (element-major rows, one contiguous piece per element) in shared memory; its warps then take the group's items,
// no barrier in between.  Item: D[element][pair] = M[element][monomial] G[pair][monomial] on the FP64 tensor cores -- A
// fragments from the staged moments, B fragments (coefficient table in fragment order) through L1 -- then the 8 x 32
// results go through a small per-warp buffer, so that lane = element: a pair's values for the elements of one geometric
// row are consecutive in CSR row (gamma, r), and a warp store covers the tile's piece of that row (the next tile, handled
// within microseconds, continues it).
__global__ void __launch_bounds__(CT_THREADS, 3)
contract_kernel(int64_t e0, int64_t e1, int64_t nnz_geo, int n_geo, const int4* __restrict__ elem_rec, unsigned int* __restrict__ ticket,
                const double* __restrict__ moments, int n_mu, const wpcd_ct_lgroup* __restrict__ lgroups, int n_lgroups,
                const wpcd_ct_item* __restrict__ items, const int32_t* __restrict__ ct_idx, const double* __restrict__ ct_g,
                const int4* __restrict__ ct_pairs, int ms_stride, int32_t* __restrict__ col_idx, double* __restrict__ values)
{
    extern __shared__ __align__(16) double ct_sm[];
    double* Ms = ct_sm;                                                   // [CT_E][ms_stride]
    double* Sw = Ms + CT_E * ms_stride + (threadIdx.x >> 5) * (8 * 33);   // this warp's [8][33] transposition buffer
    __shared__ unsigned int s_unit;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, quad = lane & 3, oct = lane >> 2;
    const int64_t n_tiles = (e1 - e0 + CT_E - 1) / CT_E;
    const uint64_t n_units = (uint64_t)n_tiles * n_lgroups;
    for (;;) {
        if (tid == 0) s_unit = atomicAdd(ticket, 1u);
        __syncthreads();
        const unsigned int u = s_unit;
        if (u >= n_units) return;
        const unsigned int tile = u / n_lgroups;
        const wpcd_ct_lgroup lg = lgroups[u - tile * n_lgroups];
        const int64_t es = e0 + (int64_t)tile * CT_E;
        const int m = (int)min((int64_t)CT_E, e1 - es);
        // ---- stage the moments of this l for the tile's elements: warp = element row, lanes along the monomials
        {
            const double* src = moments + (size_t)(es - e0) * n_mu + lg.mu_lo;
            for (int ei = warp; ei < m; ei += CT_WARPS) {
                const double* s = src + (size_t)ei * n_mu;
                double* d = Ms + ei * ms_stride;
                for (int mi = lane; mi < lg.n_mono; mi += 32) d[mi] = __ldcs(s + mi);
            }
        }
        // this lane's element: where its geometric row starts in the pattern, the row's length, its position and column
        const bool ev = lane < m;
        const int4 rec = ev ? __ldg(elem_rec + es + lane) : make_int4(0, 0, 0, 0);      // grp, cnt, gcol, row
        const int pos = (int)(es + lane - rec.x);
        __syncthreads();
        const double* r0 = Ms + min(oct, m - 1) * ms_stride;
        const double* r1 = Ms + min(8 + oct, m - 1) * ms_stride;
        const double* r2 = Ms + min(16 + oct, m - 1) * ms_stride;
        const double* r3 = Ms + min(24 + oct, m - 1) * ms_stride;
        for (int ii = lg.item_begin + warp; ii < lg.item_end; ii += CT_WARPS) {
            const wpcd_ct_item it = items[ii];
            const int kt = it.kt, np = it.n_pairs;
            const int32_t* idx = ct_idx + it.idx_off + quad;
            const double* gfr = ct_g + it.g_off + lane;        // [k][np][4]: lane (oct, quad) reads entry oct * 4 + quad = lane of step k
            const bool bl = oct < np;
            const int gstep = 4 * np;
            // lane q < np: the record of pair q (prefix of ncoupled over gamma, ncoupled(gamma), rank of gamma', gamma')
            const int4 pr = lane < np ? __ldg(ct_pairs + it.pair_off + lane) : make_int4(0, 0, 0, 0);
            const int64_t my_base = (int64_t)pr.x * nnz_geo;
            const int my_gp = pr.w * n_geo;
            double c[4][2];
#pragma unroll
            for (int j = 0; j < 4; ++j) c[j][0] = c[j][1] = 0.0;
#pragma unroll 2
            for (int k = 0; k < kt; ++k) {
                const int mi = __ldg(idx + 4 * k);
                const double b = bl ? __ldg(gfr + gstep * k) : 0.0;
                dmma_884_nv(c[0][0], c[0][1], r0[mi], b);
                dmma_884_nv(c[1][0], c[1][1], r1[mi], b);
                dmma_884_nv(c[2][0], c[2][1], r2[mi], b);
                dmma_884_nv(c[3][0], c[3][1], r3[mi], b);
            }
            // lane holds out[element 8 j + oct][pair 2 quad + h]: transpose through the warp's buffer, row = pair, lane = element
            __syncwarp();
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int j = 0; j < 4; ++j) Sw[(2 * quad + h) * 33 + 8 * j + oct] = c[j][h];
            __syncwarp();
            for (int q = 0; q < np; ++q) {
                const int64_t base = __shfl_sync(0xffffffffu, my_base, q);
                const int ncoup = __shfl_sync(0xffffffffu, pr.y, q), ci = __shfl_sync(0xffffffffu, pr.z, q);
                const int gp = __shfl_sync(0xffffffffu, my_gp, q);
                if (ev) {
                    const int64_t o = base + ((int64_t)ncoup * rec.x + (ci * rec.y + pos));
                    __stcs(values + o, Sw[q * 33 + lane]);
                    __stcs(col_idx + o, gp + rec.z);
                }
            }
        }
        __syncthreads();     // Ms is free again
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
    // contraction: staged moments [32][ms_stride] + one [8][33] transposition buffer per warp + the run's geometric columns
    const int ms_stride = ch->ct_nmono_max | 1;                 // odd: the A-fragment rows of a quarter-warp fall into different banks
    const size_t ct_smem = sizeof(double) * ((size_t)CT_E * ms_stride + (size_t)CT_WARPS * 8 * 33);
    if (ct_smem > 227 * 1024) return cudaErrorInvalidValue;
    const int n_geo = g->n_p * g->n_q;
    const int maxs = (ch->n_mu + 31) / 32;
#define WPCD_MOM2(MS, SPL)                                                                                                        \
    do {                                                                                                                      \
        err = cudaFuncSetAttribute(moments_kernel<MS, SPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mom_smem);           \
        if (err != cudaSuccess) return err;                                                                                   \
        moments_kernel<MS, SPL><<<blocks, mom_warps * 32, mom_smem, st>>>(qr, g->p_dev, g->q_dev, g->n_q, sh, e0, e1, ws.geo_col,      \
                                                                     ws.geo_row, ws.geo_phi, ch->ll_pack_dev,                 \
                                                                     ch->trip_pack_dev, ch->mu_pack_dev, ch->ab_pack_dev, ws.moments);         \
    } while (0)
#define WPCD_MOM(MS) do { if (split) WPCD_MOM2(MS, true); else WPCD_MOM2(MS, false); } while (0)
    err = cudaFuncSetAttribute(contract_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ct_smem);
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
            if (maxs <= 4) WPCD_MOM(4);
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
            // persistent CTAs pulling (tile, l-group) units from a work queue
            contract_kernel<<<ct_blocks, CT_THREADS, ct_smem, st>>>(e0, e1, nnz_geo, n_geo, ws.elem_rec, ws.counters + chunk_no, ws.moments, ch->n_mu,
                                                                    ch->ct_lgroups_dev, (int)ch->ct_lgroups.size(), ch->ct_items_dev, ch->ct_idx_dev,
                                                                    ch->ct_g_dev, ch->ct_pairs_dev, ms_stride, col_idx, values);
            ++g_launches;
            if ((err = cudaGetLastError()) != cudaSuccess) return err;
        }
    }
#undef WPCD_MOM
#undef WPCD_MOM2
    return cudaSuccess;
}

}  // namespace wpcd_detail
