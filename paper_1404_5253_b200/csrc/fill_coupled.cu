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

// Moment layout: [tile of 32 elements][mu][element in tile] (the contraction reads 32 elements of
// one monomial as one 256-byte line).
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
    const int64_t el = e - e_begin;
    double* out = moments + ((size_t)(el >> 5) * n_mu) * 32 + (el & 31);
#pragma unroll
    for (int s = 0; s < MAXS; ++s)
        if (lane + 32 * s < n_mu) out[(size_t)(lane + 32 * s) * 32] = acc[s];
}

}  // namespace

namespace {

constexpr int CT_THREADS = 256;
constexpr int CT_WARPS = CT_THREADS / 32;

__device__ __forceinline__ uint32_t smem_u32(const void* ptr) { return (uint32_t)__cvta_generic_to_shared(ptr); }

// One slab of classes, global -> shared, as a single TMA bulk copy tracked by an mbarrier.
__device__ __forceinline__ void slab_to_smem(unsigned char* dst, const unsigned char* src, uint32_t bytes, uint64_t* mbar)
{
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(mbar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(mbar)) : "memory");
    }
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(mbar)) : "memory");
}

struct TileLane {
    bool valid;
    int grp, cnt, pos, gcol;
    const double* stage;    // this warp's staged class block, [m][32], offset by the lane
};

// Asynchronous copy (cp.async, 8 bytes per lane and monomial) of one class block of a tile's moment
// row into the warp's staging buffer: it flies while the previous class is being contracted.
__device__ __forceinline__ void stage_class(const wpcd_class_desc& d, const unsigned char* slab, const double* mrow_lane,
                                            double* stage_lane)
{
    const int4* idx = reinterpret_cast<const int4*>(slab + d.idx_off);
    uint32_t dst = smem_u32(stage_lane);
    const int quads = d.nm >> 2;
#pragma unroll 2
    for (int m = 0; m < quads; ++m, dst += 1024) {
        const int4 i4 = idx[m];
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(mrow_lane + i4.x * 32) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 256), "l"(mrow_lane + i4.y * 32) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 512), "l"(mrow_lane + i4.z * 32) : "memory");
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 768), "l"(mrow_lane + i4.w * 32) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}

// All pairs of one class for the 32 elements of a warp tile.  NM = padded monomial count.
template <int NM>
__device__ __forceinline__ void contract_class(const wpcd_class_desc& d, const unsigned char* slab, const TileLane& tl,
                                               const double (&M)[NM], int64_t nnz_geo, int n_geo,
                                               int32_t* __restrict__ col_idx, double* __restrict__ values)
{
    const bool add = (d.flags & 1) != 0;
    const int4* meta = reinterpret_cast<const int4*>(slab + d.meta_off);
    const double2* G = reinterpret_cast<const double2*>(slab + d.g_off);
    const int n_pairs = d.n_pairs;
    int pi = 0;
    for (; pi + 1 < n_pairs; pi += 2) {
        const double2* g0 = G + (size_t)pi * (NM / 2);
        const double2* g1 = g0 + NM / 2;
        double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
#pragma unroll
        for (int m = 0; m < NM / 2; ++m) {
            const double2 u = g0[m], v = g1[m];
            a0 = fma(u.x, M[2 * m], a0); a1 = fma(u.y, M[2 * m + 1], a1);
            b0 = fma(v.x, M[2 * m], b0); b1 = fma(v.y, M[2 * m + 1], b1);
        }
        const int4 ma = meta[pi], mb = meta[pi + 1];
        if (tl.valid) {
            const int64_t oa = (int64_t)ma.x * nnz_geo + (int64_t)ma.y * tl.grp + (int64_t)ma.z * tl.cnt + tl.pos;
            const int64_t ob = (int64_t)mb.x * nnz_geo + (int64_t)mb.y * tl.grp + (int64_t)mb.z * tl.cnt + tl.pos;
            values[oa] = add ? values[oa] + (a0 + a1) : a0 + a1; col_idx[oa] = ma.w * n_geo + tl.gcol;
            values[ob] = add ? values[ob] + (b0 + b1) : b0 + b1; col_idx[ob] = mb.w * n_geo + tl.gcol;
        }
    }
    if (pi < n_pairs) {
        const double2* g0 = G + (size_t)pi * (NM / 2);
        double a0 = 0.0, a1 = 0.0;
#pragma unroll
        for (int m = 0; m < NM / 2; ++m) { const double2 u = g0[m]; a0 = fma(u.x, M[2 * m], a0); a1 = fma(u.y, M[2 * m + 1], a1); }
        const int4 ma = meta[pi];
        if (tl.valid) {
            const int64_t oa = (int64_t)ma.x * nnz_geo + (int64_t)ma.y * tl.grp + (int64_t)ma.z * tl.cnt + tl.pos;
            values[oa] = add ? values[oa] + (a0 + a1) : a0 + a1; col_idx[oa] = ma.w * n_geo + tl.gcol;
        }
    }
}

// slab_tab[s] = (blob offset, bytes, first CTA, CTA count)
__global__ void __launch_bounds__(CT_THREADS, 2)
contract_kernel(int64_t e_begin, int64_t e_end, int64_t nnz_geo, int n_geo, const int32_t* __restrict__ geo_col,
                const int32_t* __restrict__ geo_row, const int32_t* __restrict__ geo_row_ptr,
                const double* __restrict__ moments, int n_mu, const unsigned char* __restrict__ slab_blob,
                const int4* __restrict__ slab_tab, int n_slabs, int stage_off, int32_t* __restrict__ col_idx,
                double* __restrict__ values)
{
    extern __shared__ __align__(128) unsigned char slab[];
    __shared__ __align__(8) uint64_t mbar;
    int s = 0;
    while (s + 1 < n_slabs && (int)blockIdx.x >= slab_tab[s + 1].z) ++s;
    const int4 st = slab_tab[s];
    slab_to_smem(slab, slab_blob + st.x, (uint32_t)st.y, &mbar);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_classes = reinterpret_cast<const wpcd_slab_header*>(slab)->n_classes;
    const wpcd_class_desc* desc = reinterpret_cast<const wpcd_class_desc*>(slab + sizeof(wpcd_slab_header));
    const int64_t n_tiles = (e_end - e_begin + 31) / 32;
    const int64_t warps_here = (int64_t)st.w * CT_WARPS;
    // staging buffers behind the slab: [warp][32 monomials][32 lanes]
    double* stage_lane = reinterpret_cast<double*>(slab + stage_off) + (size_t)warp * (WPCD_MAX_NM * 32) + lane;
    int64_t tile = (int64_t)((int)blockIdx.x - st.z) * CT_WARPS + warp;
    if (tile < n_tiles && n_classes > 0) stage_class(desc[0], slab, moments + (size_t)tile * n_mu * 32 + lane, stage_lane);
    for (; tile < n_tiles; tile += warps_here) {
        const int64_t e = e_begin + tile * 32 + lane;
        TileLane tl;
        tl.valid = e < e_end;
        const int64_t ec = tl.valid ? e : e_end - 1;      // idle lanes shadow the last element (loads stay in range)
        const int r = geo_row[ec];
        tl.gcol = geo_col[ec];
        tl.grp = geo_row_ptr[r];
        tl.cnt = geo_row_ptr[r + 1] - tl.grp;
        tl.pos = (int)(ec - tl.grp);
        tl.stage = stage_lane;
        const double* mrow_lane = moments + (size_t)tile * n_mu * 32 + lane;
        for (int ci = 0; ci < n_classes; ++ci) {
            const wpcd_class_desc d = desc[ci];
            // the block of class ci has been copied to the staging buffer: move it to registers, then let
            // the copy of the next block (next class, or first class of this warp's next tile) fly
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
#define WPCD_CT(NMV)                                                                                              \
    {                                                                                                             \
        double M[NMV];                                                                                            \
        _Pragma("unroll") for (int m = 0; m < NMV; ++m) M[m] = stage_lane[m * 32];                                \
        __syncwarp();                                                                                             \
        if (ci + 1 < n_classes) stage_class(desc[ci + 1], slab, mrow_lane, stage_lane);                           \
        else if (tile + warps_here < n_tiles)                                                                     \
            stage_class(desc[0], slab, moments + (size_t)(tile + warps_here) * n_mu * 32 + lane, stage_lane);      \
        contract_class<NMV>(d, slab, tl, M, nnz_geo, n_geo, col_idx, values);                                     \
    }
            switch (d.nm) {
            case 4: WPCD_CT(4) break;
            case 8: WPCD_CT(8) break;
            case 12: WPCD_CT(12) break;
            case 16: WPCD_CT(16) break;
            case 20: WPCD_CT(20) break;
            case 24: WPCD_CT(24) break;
            case 28: WPCD_CT(28) break;
            default: WPCD_CT(32) break;
            }
#undef WPCD_CT
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
    static const int g_forced = [] { const char* e = getenv("WPCD_MOM_G"); return e ? atoi(e) : 0; }();   // tuning knob
    sh.n = n_quad; sh.NS = split ? std::max(n_quad, 4 * SPLIT_MAX_U) : n_quad; sh.G = std::max(1, std::min(32 / n_quad, g_forced > 0 ? g_forced : (n_quad <= 8 ? 4 : 2)));   // measured: n = 8: 4 beats 2 by 13 %, n = 10: 3 loses to 2
    sh.K1 = ch->k_max + 1; sh.SP = 8 * ((sh.K1 + 7) / 8) + 4;
    sh.ST = 8 * ((ch->n_ll + 7) / 8) + 4; sh.IS = 8 * ((ch->n_ll + 7) / 8) + 2;
    sh.LM1 = ch->l_max + 1; sh.CP = 2 * ch->l_max + 3; sh.n_ab = ch->n_ab;
    sh.n_ll = ch->n_ll; sh.n_trip = ch->n_trip; sh.n_mu = ch->n_mu;
    if ((sh.SP - 4) * sh.IS >= 65536) return cudaErrorInvalidValue;
    const int mom_warps = MOM_MAX_WARPS;
    const size_t mom_smem = sizeof(double) * ((size_t)((((sh.LM1 * sh.LM1 + sh.n_trip + 1) >> 1) + 1) & ~1) + (size_t)mom_warps * moment_smem_doubles(sh));
    size_t ct_smem = 0;
    double cost_sum = 0.0;
    for (auto& sl : ch->slabs) { ct_smem = std::max(ct_smem, sl.bytes); cost_sum += sl.cost; }
    const int stage_off = (int)((ct_smem + 127) & ~(size_t)127);
    ct_smem = (size_t)stage_off + sizeof(double) * CT_WARPS * WPCD_MAX_NM * 32;
    if (ct_smem > 227 * 1024 || mom_smem > 227 * 1024) return cudaErrorInvalidValue;
    // CTAs per slab in proportion to its cost, two CTAs per SM per pass
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int n_slabs = (int)ch->slabs.size();
    int n_pass = 0;
    for (auto& sl : ch->slabs) n_pass = std::max(n_pass, sl.pass + 1);
    std::vector<int4> tab(n_slabs);
    std::vector<int> pass_first(n_pass + 1, 0), pass_ctas(n_pass, 0);
    for (int pass = 0, s = 0; pass < n_pass; ++pass) {       // slabs are stored pass by pass
        double cost_pass = 0.0;
        pass_first[pass] = s;
        for (int t = s; t < n_slabs && ch->slabs[t].pass == pass; ++t) cost_pass += ch->slabs[t].cost;
        for (; s < n_slabs && ch->slabs[s].pass == pass; ++s) {
            int cnt = std::max(1, (int)llround(2.0 * sms * ch->slabs[s].cost / std::max(cost_pass, 1.0)));
            tab[s] = make_int4((int)ch->slabs[s].offset, (int)ch->slabs[s].bytes, pass_ctas[pass], cnt);
            pass_ctas[pass] += cnt;
        }
        pass_first[pass + 1] = s;
    }
    (void)cost_sum;
    int4* tab_dev = reinterpret_cast<int4*>(ws.slab_tab);
    err = cudaMemcpyAsync(tab_dev, tab.data(), sizeof(int4) * n_slabs, cudaMemcpyHostToDevice, st);
    if (err != cudaSuccess) return err;
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
    for (int64_t e0 = 0; e0 < nnz_geo; e0 += ws.chunk) {
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
            for (int pass = 0; pass < n_pass; ++pass) {
                contract_kernel<<<pass_ctas[pass], CT_THREADS, ct_smem, st>>>(e0, e1, nnz_geo, n_geo, ws.geo_col, ws.geo_row, geo_row_ptr,
                                                                              ws.moments, ch->n_mu, ch->slab_blob_dev,
                                                                              tab_dev + pass_first[pass],
                                                                              pass_first[pass + 1] - pass_first[pass], stage_off, col_idx, values);
                ++g_launches;
                if ((err = cudaGetLastError()) != cudaSuccess) return err;
            }
        }
    }
#undef WPCD_MOM
#undef WPCD_MOM2
    return cudaSuccess;
}

}  // namespace wpcd_detail
