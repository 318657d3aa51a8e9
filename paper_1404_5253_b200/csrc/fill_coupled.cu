// fill_coupled.cu -- paper step 3 for coupled channels (configs 3-5):
// value[gamma,gamma'] = norm * sum_{k,l1,l1'} g * integral of F P_k(x) cos^{A+1} sin^{B+1} /
// (zeta1^{l'+1} zeta2^{l+1}) over (phi, x), (A15) with reading R1 (A = l1+l1',
// B = l+l'-A).  The geometry (F, zeta, limits) is shared by ALL channel pairs of a geometric
// element, so the work is split in two kernels:
//
//   moments_kernel   one warp per geometric element: monomial moments
//                      M[mu] = norm * sum_nodes w F P_k(x) cos^{A+1} sin^{B+1} zeta1^{-(l'+1)} zeta2^{-(l+1)}
//                    for the n_mu distinct mu = (k, A, l, l') of the channel set (152 .. 524),
//                    written to a scratch block [element][mu].
//   contract_kernel  one CTA per tile of 32 consecutive geometric elements: the moment tile is
//                    staged in shared memory ([mu][33] doubles), the (g, mu) term lists of the
//                    coupled pairs stream through shared memory in groups, lane = element, and
//                    every pair writes 32 consecutive CSR values + column indices (coalesced).
#include <math.h>

#include <algorithm>

#include "quad_device.cuh"
#include "wpcd_internal.h"

using namespace wpcd_quad;

namespace {

__constant__ double k_xi[WPCD_MAX_QUAD];
__constant__ double k_w[WPCD_MAX_QUAD];

constexpr int MOM_WARPS = 4;

__device__ __forceinline__ double ipow(double b, int e)
{
    double r = 1.0;
    for (int i = 0; i < e; ++i) r *= b;
    return r;
}

// packed monomial: k | A<<8 | l<<16 | l'<<24
template <int MAXS>
__global__ void __launch_bounds__(MOM_WARPS * 32)
moments_kernel(const double* __restrict__ p, const double* __restrict__ q, int n_q, int n,
               int64_t e_begin, int64_t e_end, const int32_t* __restrict__ geo_col, const int32_t* __restrict__ geo_row,
               const double2* __restrict__ geo_phi, const wpcd_monomial* __restrict__ mu_tab, int n_mu, int K1, int LP, int CP,
               double* __restrict__ moments)
{
    extern __shared__ double sm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t e = e_begin + (int64_t)blockIdx.x * MOM_WARPS + warp;
    if (e >= e_end) return;
    const int per_warp = n * (1 + K1 + 2 * LP) + 2 * CP;
    double* wF = sm + (size_t)warp * per_warp;   // [n]
    double* Pk = wF + n;                         // [n][K1]
    double* z1p = Pk + n * K1;                   // [n][LP]   (1/zeta1)^e
    double* z2p = z1p + n * LP;                  // [n][LP]
    double* cpw = z2p + n * LP;                  // [CP]      cos^e
    double* spw = cpw + CP;                      // [CP]      sin^e

    int packed[MAXS];
    double acc[MAXS];
#pragma unroll
    for (int s = 0; s < MAXS; ++s) {
        const int m = lane + 32 * s;
        acc[s] = 0.0;
        packed[s] = 0;
        if (m < n_mu) {
            const wpcd_monomial t = mu_tab[m];
            packed[s] = (int)t.k | ((int)t.A << 8) | ((int)t.l << 16) | ((int)t.lp << 24);
        }
    }
    const int col = geo_col[e], row = geo_row[e];
    const double2 ph = geo_phi[e];
    const Cell z = load_cell(p, q, n_q, row, col);
    const double norm = cell_norm(z);
    const double half_phi = 0.5 * (ph.y - ph.x), mid_phi = 0.5 * (ph.x + ph.y);
    if (ph.x < ph.y) {
        for (int m = 0; m < n; ++m) {
            PhiNode s;
            if (!phi_node(z, mid_phi + half_phi * k_xi[m], s)) continue;   // warp-uniform
            const double half_u = 0.5 * (s.u_hi - s.u_lo), mid_u = 0.5 * (s.u_lo + s.u_hi);
            const double wphi = half_phi * k_w[m] * half_u * norm;
            if (lane < CP) { cpw[lane] = ipow(s.C, lane); spw[lane] = ipow(s.S, lane); }
            for (int r = lane; r < n; r += 32) {
                const double u = mid_u + half_u * k_xi[r];
                const double x = u - 1.0;
                const double iz1 = rsqrt(s.b1 + s.beta * u), iz2 = rsqrt(s.b2 + s.beta * u);
                wF[r] = wphi * k_w[r] * F_A14(z, s, iz1, iz2);
                double p0 = 1.0, p1 = x;
                Pk[r * K1] = 1.0;
                if (K1 > 1) Pk[r * K1 + 1] = x;
                for (int k = 2; k < K1; ++k) {
                    const double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
                    Pk[r * K1 + k] = p2;
                    p0 = p1; p1 = p2;
                }
                double a1 = 1.0, a2 = 1.0;
                for (int ex = 0; ex < LP; ++ex) {
                    z1p[r * LP + ex] = a1; z2p[r * LP + ex] = a2;
                    a1 *= iz1; a2 *= iz2;
                }
            }
            __syncwarp();
#pragma unroll
            for (int sl = 0; sl < MAXS; ++sl) {
                if (lane + 32 * sl < n_mu) {
                    const int pk = packed[sl];
                    const int k = pk & 0xff, A = (pk >> 8) & 0xff, l = (pk >> 16) & 0xff, lp = (pk >> 24) & 0xff;
                    double inner = 0.0;
                    for (int r = 0; r < n; ++r)
                        inner = fma(wF[r] * Pk[r * K1 + k], z1p[r * LP + lp + 1] * z2p[r * LP + l + 1], inner);
                    acc[sl] = fma(cpw[A + 1] * spw[l + lp - A + 1], inner, acc[sl]);
                }
            }
            __syncwarp();
        }
    }
    double* out = moments + (size_t)(e - e_begin) * n_mu;
#pragma unroll
    for (int sl = 0; sl < MAXS; ++sl)
        if (lane + 32 * sl < n_mu) out[lane + 32 * sl] = acc[sl];
}

}  // namespace

namespace {

constexpr int CT_THREADS = 256;
constexpr int CT_WARPS = CT_THREADS / 32;
constexpr int TILE = 32;
constexpr int MS_LD = TILE + 1;   // padded leading dimension of the moment tile

__global__ void __launch_bounds__(CT_THREADS)
contract_kernel(int64_t e_begin, int64_t e_end, int64_t nnz_geo, int n_geo, const int32_t* __restrict__ geo_col,
                const int32_t* __restrict__ geo_row, const int32_t* __restrict__ geo_row_ptr,
                const double* __restrict__ moments, int n_mu, int n_pairs, int pair_group, int stage_cap,
                const int32_t* __restrict__ mterm_ptr, const int32_t* __restrict__ mterm_mu, const double* __restrict__ mterm_g,
                const int32_t* __restrict__ pair_gamma, const int32_t* __restrict__ pair_gammap, const int32_t* __restrict__ pair_ci,
                const int32_t* __restrict__ ncoupled, const int64_t* __restrict__ chan_off,
                int32_t* __restrict__ col_idx, double* __restrict__ values)
{
    extern __shared__ double sm[];
    double* Ms = sm;                                   // [n_mu][MS_LD]
    double* sg = Ms + (size_t)n_mu * MS_LD;            // [stage_cap]
    int32_t* smu = reinterpret_cast<int32_t*>(sg + stage_cap);   // [stage_cap]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t tile0 = e_begin + (int64_t)blockIdx.x * TILE;
    const int n_here = (int)min((int64_t)TILE, e_end - tile0);

    // moment tile: global [element][mu] -> shared [mu][element]
    for (int idx = threadIdx.x; idx < TILE * n_mu; idx += CT_THREADS) {
        const int el = idx / n_mu, m = idx - el * n_mu;
        Ms[m * MS_LD + el] = el < n_here ? moments[(size_t)(tile0 - e_begin + el) * n_mu + m] : 0.0;
    }
    // this lane's element
    const bool valid = lane < n_here;
    int64_t grp = 0, cnt = 0, pos = 0;
    int gcol = 0;
    if (valid) {
        const int64_t e = tile0 + lane;
        const int r = geo_row[e];
        gcol = geo_col[e];
        grp = geo_row_ptr[r];
        cnt = geo_row_ptr[r + 1] - grp;
        pos = e - grp;
    }
    for (int c0 = 0; c0 < n_pairs; c0 += pair_group) {
        const int c1 = min(n_pairs, c0 + pair_group);
        const int t0 = mterm_ptr[c0], t1 = mterm_ptr[c1];
        __syncthreads();                                // previous group consumed / Ms complete
        for (int t = t0 + threadIdx.x; t < t1; t += CT_THREADS) { sg[t - t0] = mterm_g[t]; smu[t - t0] = mterm_mu[t]; }
        __syncthreads();
        for (int c = c0 + warp; c < c1; c += CT_WARPS) {
            const int ta = mterm_ptr[c] - t0, tb = mterm_ptr[c + 1] - t0;
            double acc = 0.0;
            for (int t = ta; t < tb; ++t) acc = fma(sg[t], Ms[smu[t] * MS_LD + lane], acc);
            if (valid) {
                const int ga = pair_gamma[c];
                const int64_t out = chan_off[ga] * nnz_geo + (int64_t)ncoupled[ga] * grp + (int64_t)pair_ci[c] * cnt + pos;
                values[out] = acc;
                col_idx[out] = pair_gammap[c] * n_geo + gcol;
            }
        }
    }
}

}  // namespace

namespace wpcd_detail {

cudaError_t launch_fill_coupled(const wpcd_grid* g, const wpcd_channels* ch, int n_quad, const double* xi, const double* w,
                                int64_t nnz_geo, const Workspace& ws, const int64_t* /*row_ptr*/, const int32_t* geo_row_ptr,
                                int32_t* col_idx, double* values, cudaStream_t st)
{
    cudaError_t err = cudaMemcpyToSymbolAsync(k_xi, xi, sizeof(double) * n_quad, 0, cudaMemcpyHostToDevice, st);
    if (err != cudaSuccess) return err;
    err = cudaMemcpyToSymbolAsync(k_w, w, sizeof(double) * n_quad, 0, cudaMemcpyHostToDevice, st);
    if (err != cudaSuccess) return err;
    if (nnz_geo == 0 || ch->n_pairs == 0) return cudaSuccess;
    const int n_mu = ch->n_mu, K1 = ch->k_max + 1, LP = ch->l_max + 2, CP = 2 * ch->l_max + 2;
    if (CP > 32 || n_mu > 32 * 32) return cudaErrorInvalidValue;
    // moments kernel shared memory
    const size_t mom_smem = sizeof(double) * (size_t)MOM_WARPS * ((size_t)n_quad * (1 + K1 + 2 * LP) + 2 * CP);
    // contraction kernel: pair group so that moment tile + staged terms fit
    const size_t ms_bytes = sizeof(double) * (size_t)n_mu * MS_LD;
    int pair_group = 128, stage_cap = 0;
    for (;; pair_group /= 2) {
        stage_cap = 0;
        for (int c0 = 0; c0 < ch->n_pairs; c0 += pair_group) {
            int c1 = std::min(ch->n_pairs, c0 + pair_group);
            stage_cap = std::max(stage_cap, ch->mterm_ptr[c1] - ch->mterm_ptr[c0]);
        }
        stage_cap = (stage_cap + 1) & ~1;
        if (ms_bytes + 12 * (size_t)stage_cap <= 200 * 1024 || pair_group == 1) break;
    }
    const size_t ct_smem = ms_bytes + 12 * (size_t)stage_cap;
    if (ct_smem > 227 * 1024 || mom_smem > 227 * 1024) return cudaErrorInvalidValue;
    const int n_geo = g->n_p * g->n_q;
    const int maxs = (n_mu + 31) / 32;
#define WPCD_MOM(MS)                                                                                                          \
    do {                                                                                                                      \
        err = cudaFuncSetAttribute(moments_kernel<MS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mom_smem);           \
        if (err != cudaSuccess) return err;                                                                                   \
        moments_kernel<MS><<<blocks, MOM_WARPS * 32, mom_smem, st>>>(g->p_dev, g->q_dev, g->n_q, n_quad, e0, e1, ws.geo_col,  \
                                                                     ws.geo_row, ws.geo_phi, ch->mu_dev, n_mu, K1, LP, CP,    \
                                                                     ws.moments);                                             \
    } while (0)
    err = cudaFuncSetAttribute(contract_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ct_smem);
    if (err != cudaSuccess) return err;
    for (int64_t e0 = 0; e0 < nnz_geo; e0 += ws.chunk) {
        const int64_t e1 = std::min(nnz_geo, e0 + ws.chunk);
        {
            const unsigned blocks = (unsigned)((e1 - e0 + MOM_WARPS - 1) / MOM_WARPS);
            StageTimer timer(WPCD_STAGE_MOMENTS, st);
            if (maxs <= 4) WPCD_MOM(4);
            else if (maxs <= 8) WPCD_MOM(8);
            else if (maxs <= 12) WPCD_MOM(12);
            else if (maxs <= 16) WPCD_MOM(16);
            else if (maxs <= 20) WPCD_MOM(20);
            else if (maxs <= 24) WPCD_MOM(24);
            else WPCD_MOM(32);
            ++g_launches;
            if ((err = cudaGetLastError()) != cudaSuccess) return err;
        }
        {
            const unsigned blocks = (unsigned)((e1 - e0 + TILE - 1) / TILE);
            StageTimer timer(WPCD_STAGE_CONTRACT, st);
            contract_kernel<<<blocks, CT_THREADS, ct_smem, st>>>(e0, e1, nnz_geo, n_geo, ws.geo_col, ws.geo_row, geo_row_ptr, ws.moments,
                                                                 n_mu, ch->n_pairs, pair_group, stage_cap, ch->mterm_ptr_dev,
                                                                 ch->mterm_mu_dev, ch->mterm_g_dev, ch->pair_gamma_dev,
                                                                 ch->pair_gammap_dev, ch->pair_ci_dev, ch->ncoupled_dev, ch->chan_off_dev,
                                                                 col_idx, values);
            ++g_launches;
            if ((err = cudaGetLastError()) != cudaSuccess) return err;
        }
    }
#undef WPCD_MOM
    return cudaSuccess;
}

}  // namespace wpcd_detail
