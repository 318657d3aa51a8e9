// spmv_blocked.cu -- y = P0 x through the block structure of P0 (the sparse product of step 5).
//
// P0 = (channel coupling mask) x (geometric pattern): CSR row (gamma, r) holds, for every gamma' coupled to gamma in
// ascending order, the SAME cnt(r) geometric columns c_s shifted by gamma' n_geo, stored
// [gamma' rank t][geometric entry s].  So all n_ch rows of one geometric row r read the same n_ch x cnt values of x.
// One CTA takes a geometric row: it gathers X[gamma'][s] = x[gamma' n_geo + c_s] into shared memory ONCE (n_ch x cnt
// gathers instead of one per nonzero: the gathers of the general CSR product drop by the number of coupled channels),
// and its warps then stream ONLY the values of the rows (gamma, r), gamma = 0 .. n_ch-1: 8 bytes per nonzero from HBM
// instead of 12, no column index is read beyond the cnt entries that give c_s.  With X stored at stride cnt, the entries
// of a row that belong to a RUN of consecutive gamma' are a plain dot product of two contiguous arrays (values from
// global memory, X from shared memory): no index arithmetic per entry.  Geometric rows are dealt heaviest region first
// through a work queue (row lengths are very skewed and grow with the cell indices).
#include <algorithm>
#include <atomic>
#include <mutex>

#include "wpcd_internal.h"

namespace {

template <int NV> struct GbUnroll { static constexpr int value = NV >= 4 ? 4 : 8; };   // 32-entry batches of one segment whose value loads are issued together
constexpr int GB_RING = 64;          // work-queue slots (concurrent launches)

__device__ unsigned int g_queue[GB_RING][2];     // (next geometric row, CTAs done); the last CTA of a launch resets its slot

// acc[v] += sum_i V[i] X[v * xs + i], i = 0 .. len-1, lanes strided; the value loads of GB_UNR batches in flight together
// (one plane of X per vector: consecutive lanes read consecutive doubles, no bank conflicts)
template <int NV>
__device__ __forceinline__ void segment_dot(const double* __restrict__ V, const double* __restrict__ X, int xs, int len, int lane, double (&acc)[NV])
{
    constexpr int GB_UNR = GbUnroll<NV>::value;
    for (int i0 = lane; i0 < len; i0 += 32 * GB_UNR) {
        double a[GB_UNR];
#pragma unroll
        for (int k = 0; k < GB_UNR; ++k) a[k] = i0 + 32 * k < len ? __ldcs(V + i0 + 32 * k) : 0.0;
#pragma unroll
        for (int k = 0; k < GB_UNR; ++k) {
            const int i = i0 + 32 * k;
            if (i < len) {
#pragma unroll
                for (int v = 0; v < NV; ++v) acc[v] = fma(a[k], X[v * xs + i], acc[v]);
            }
        }
    }
}

// The same with a software pipeline (the next batch's values are requested before this batch is multiplied): pays for two
// vectors (4.8 against 5.7 ms on the 3.2e9-nonzero matrix), costs registers and CTAs per SM for one.
template <int NV>
__device__ __forceinline__ void segment_dot_pipelined(const double* __restrict__ V, const double* __restrict__ X, int xs, int len, int lane,
                                                      double (&acc)[NV])
{
    constexpr int GB_UNR = GbUnroll<NV>::value;
    double a[GB_UNR], a2[GB_UNR];
#pragma unroll
    for (int k = 0; k < GB_UNR; ++k) a[k] = lane + 32 * k < len ? __ldcs(V + lane + 32 * k) : 0.0;
    for (int i0 = lane; i0 < len; i0 += 32 * GB_UNR) {
        const int n0 = i0 + 32 * GB_UNR;
#pragma unroll
        for (int k = 0; k < GB_UNR; ++k) a2[k] = n0 + 32 * k < len ? __ldcs(V + n0 + 32 * k) : 0.0;
#pragma unroll
        for (int k = 0; k < GB_UNR; ++k) {
            const int i = i0 + 32 * k;
            if (i < len) {
#pragma unroll
                for (int v = 0; v < NV; ++v) acc[v] = fma(a[k], X[v * xs + i], acc[v]);
            }
        }
#pragma unroll
        for (int k = 0; k < GB_UNR; ++k) a[k] = a2[k];
    }
}

template <int NV>
__device__ __forceinline__ void segment(const double* __restrict__ V, const double* __restrict__ X, int xs, int len, int lane, double (&acc)[NV])
{
    if (NV == 2) segment_dot_pipelined<NV>(V, X, xs, len, lane, acc);
    else segment_dot<NV>(V, X, xs, len, lane, acc);
}

// x, y: NV vectors, vector-major (x[v * ldx + column]).  cap: doubles of the X tile per vector.
template <int NV, int GB_THREADS>
__global__ void __launch_bounds__(GB_THREADS)
spmv_georow_kernel(int n_geo, int n_ch, const int32_t* __restrict__ geo_row_ptr, const int32_t* __restrict__ col_idx,
                   const double* __restrict__ values, const int64_t* __restrict__ chan_off, const int32_t* __restrict__ ncoupled,
                   const int32_t* __restrict__ run_ptr, const int4* __restrict__ runs, int first_gamma, int first_gp,
                   const double* __restrict__ x, double* __restrict__ y, int64_t ldx, int cap, int slot)
{
    extern __shared__ __align__(16) double gb_sm[];
    double* X = gb_sm;                                         // [NV][channels of the chunk][cs]
    double* ysum = X + (size_t)cap * NV;                       // [n_ch][NV]
    int32_t* gcol = reinterpret_cast<int32_t*>(ysum + (size_t)n_ch * NV);      // [cs]
    __shared__ unsigned int s_row;
    constexpr int GB_WARPS = GB_THREADS / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t nnz_geo = geo_row_ptr[n_geo];
    for (;;) {
        if (tid == 0) s_row = atomicAdd(&g_queue[slot][0], 1u);
        __syncthreads();
        const unsigned int ticket = s_row;
        if (ticket >= (unsigned int)n_geo) break;
        const int r = n_geo - 1 - (int)ticket;                 // the long rows sit at the high cell indices: they go first
        const int grp = geo_row_ptr[r], cnt = geo_row_ptr[r + 1] - grp;
        for (int i = tid; i < n_ch * NV; i += GB_THREADS) ysum[i] = 0.0;
        if (cnt > 0 && first_gamma >= 0) {
            // the geometric columns of the row: block t = 0 of the first channel that has entries
            const int32_t* c0 = col_idx + (chan_off[first_gamma] * nnz_geo + (int64_t)ncoupled[first_gamma] * grp);
            const int S = min(cnt, cap);                       // geometric entries per chunk (all of them unless the row is huge)
            for (int s0 = 0; s0 < cnt; s0 += S) {
                const int cs = min(S, cnt - s0);
                const int gpc = max(1, cap / cs);              // channels per chunk
                __syncthreads();                               // the previous chunk's gcol is no longer read
                for (int s = tid; s < cs; s += GB_THREADS) gcol[s] = __ldg(c0 + s0 + s) - first_gp * n_geo;
                for (int glo = 0; glo < n_ch; glo += gpc) {
                    const int ghi = min(n_ch, glo + gpc);
                    __syncthreads();                           // gcol is there; the previous X tile is no longer read
                    {
                        // tile entry i = (channel gg, geometric entry s), advanced without divisions
                        const int n_tile = (ghi - glo) * cs;
                        const int dq = GB_THREADS / cs, dr = GB_THREADS - dq * cs;
                        int gg = tid / cs, s = tid - gg * cs;
                        for (int i = tid; i < n_tile; i += GB_THREADS) {
                            const double* xp = x + (int64_t)(glo + gg) * n_geo + gcol[s];
#pragma unroll
                            for (int v = 0; v < NV; ++v) X[v * cap + i] = __ldg(xp + v * ldx);
                            gg += dq; s += dr;
                            if (s >= cs) { s -= cs; ++gg; }
                        }
                    }
                    __syncthreads();
                    for (int ga = warp; ga < n_ch; ga += GB_WARPS) {
                        const int nc = ncoupled[ga];
                        if (nc == 0) continue;
                        const double* vrow = values + (chan_off[ga] * nnz_geo + (int64_t)nc * grp);
                        double acc[NV];
#pragma unroll
                        for (int v = 0; v < NV; ++v) acc[v] = 0.0;
                        bool any = false;
                        for (int ri = run_ptr[ga]; ri < run_ptr[ga + 1]; ++ri) {
                            const int4 run = __ldg(runs + ri);              // (rank of the first, first gamma', length)
                            const int a0 = max(run.y, glo), a1 = min(run.y + run.z, ghi);     // channels of the run inside the chunk
                            if (a0 >= a1) continue;
                            any = true;
                            const int t0 = run.x + (a0 - run.y);
                            if (cs == cnt) {
                                segment<NV>(vrow + (int64_t)t0 * cnt, X + (a0 - glo) * cs, cap, (a1 - a0) * cnt, lane, acc);
                            } else {
                                for (int j = 0; j < a1 - a0; ++j)
                                    segment<NV>(vrow + (int64_t)(t0 + j) * cnt + s0, X + (a0 - glo + j) * cs, cap, cs, lane, acc);
                            }
                        }
                        if (!any) continue;
#pragma unroll
                        for (int v = 0; v < NV; ++v) {
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) acc[v] += __shfl_xor_sync(0xffffffffu, acc[v], o);
                        }
                        if (lane == 0) {
#pragma unroll
                            for (int v = 0; v < NV; ++v) ysum[ga * NV + v] += acc[v];
                        }
                    }
                }
            }
        }
        __syncthreads();
        for (int i = tid; i < n_ch * NV; i += GB_THREADS) {
            const int ga = i / NV, v = i - ga * NV;
            y[v * ldx + (int64_t)ga * n_geo + r] = ysum[i];
        }
    }
    // the last CTA of the launch puts the queue slot back to zero
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(&g_queue[slot][1], 1u) == gridDim.x - 1) {
            g_queue[slot][0] = 0u;
            g_queue[slot][1] = 0u;
            __threadfence();
        }
    }
}

// 8-byte load of a matrix value that asks L2 to bring the whole 256-byte neighbourhood from DRAM: the A-fragment loads below
// touch 32 bytes per row at a time (7.40 -> 7.15 ms on the 3.2e9-nonzero matrix)
__device__ __forceinline__ double ld_value_l2_256(const double* p)
{
    double v;
    asm volatile("ld.global.nc.L2::256B.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}

__device__ __forceinline__ void dmma_884g(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---------------------------------------------------------------------------------------------------------------
// Eight vectors per pass on the FP64 tensor cores.  For a fixed geometric row all n_ch rows (gamma, r) use the same
// tile X[gamma'][s]; indexed by the TILE entry i = (gamma', s), row gamma holds the value V_gamma[rank_gamma(gamma') cnt + s]
// (or none, if gamma' is not coupled to gamma).  So 8 rows x 4 tile entries x 8 vectors is one MMA:
//   D[row][vector] += A[row][entry] B[entry][vector],  A = values (each lane loads one value of ITS row), B = X planes.
// A value is loaded once and used for 8 vectors, a tile word is read once per 8 rows: 1 byte of shared memory per
// multiply-add instead of 8 (the scalar kernel above is bound by exactly that for 8 vectors).
// Warps: a CTA has 8 ROW GROUPS of 8 consecutive channels x (16 / groups) warps per group, which share the group's gamma' range;
// accumulators stay in registers over all chunks of the geometric row and are summed in a fixed order at its end.
// xi[c][v] = x[v][c]: the 8 vectors interleaved, so that the tile of a geometric row is gathered in 64-byte pieces
__global__ void __launch_bounds__(256)
interleave8_kernel(int64_t rows, int nv, const double* __restrict__ x, int64_t ldx, double* __restrict__ xi)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= rows) return;
    double v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = k < nv ? __ldg(x + k * ldx + c) : 0.0;
    double4* o = reinterpret_cast<double4*>(xi + c * 8);
    o[0] = make_double4(v[0], v[1], v[2], v[3]);
    o[1] = make_double4(v[4], v[5], v[6], v[7]);
}

constexpr int GM_THREADS = 512;
constexpr int GM_WARPS = GM_THREADS / 32;
constexpr int GM_GROUPS = 8;                        // at most 8 row groups per CTA: channels 8 g .. 8 g + 7 (n_ch <= 64)
constexpr int GM_UNR = 8;

__global__ void __launch_bounds__(GM_THREADS, 1)
spmv_georow_mma8_kernel(int n_geo, int n_ch, const int32_t* __restrict__ geo_row_ptr, const int32_t* __restrict__ col_idx,
                        const double* __restrict__ values, const int64_t* __restrict__ chan_off, const int32_t* __restrict__ ncoupled,
                        const int32_t* __restrict__ run_ptr, const int4* __restrict__ runs, int first_gamma, int first_gp,
                        const double* __restrict__ xi, double* __restrict__ y, int64_t ldx, int nv, int cap, int slot)
{
    extern __shared__ __align__(16) double gb_sm[];
    const int ps = cap + 4;                                                // plane stride = 4 (mod 16): the B fragments of a quarter-warp fall into different banks
    double* X = gb_sm;                                                     // [8 vectors][channels of the chunk][cs], planes ps apart
    double* ypart = X + (size_t)ps * 8;                                   // [warp][8 rows][8 vectors]
    int32_t* gcol = reinterpret_cast<int32_t*>(ypart + GM_WARPS * 64);   // [cap]
    int32_t* rank_tab = gcol + cap;                                        // [n_ch][n_ch]: rank of gamma' in row gamma, or -1
    __shared__ unsigned int s_row;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, quad = lane & 3, oct = lane >> 2;
    const int n_grp = max(1, (n_ch + 7) >> 3), wpg = GM_WARPS / n_grp;             // row groups in use, warps per row group
    const int grp_id = warp / wpg, wig = warp - grp_id * wpg;              // row group, warp inside the group (the warps left over idle)
    const int my_row = grp_id * 8 + oct;                                   // this lane's channel (A fragment row)
    const int64_t nnz_geo = geo_row_ptr[n_geo];
    // rank table from the runs of consecutive coupled channels
    for (int i = tid; i < n_ch * n_ch; i += GM_THREADS) rank_tab[i] = -1;
    __syncthreads();
    for (int ga = warp; ga < n_ch; ga += GM_THREADS / 32)
        for (int ri = run_ptr[ga]; ri < run_ptr[ga + 1]; ++ri) {
            const int4 run = __ldg(runs + ri);                             // (rank of the first, first gamma', length)
            for (int j = lane; j < run.z; j += 32) rank_tab[ga * n_ch + run.y + j] = run.x + j;
        }
    const bool row_ok = grp_id < n_grp && my_row < n_ch;
    const int my_nc = row_ok ? ncoupled[my_row] : 0;
    const int64_t my_off = row_ok ? chan_off[my_row] * nnz_geo : 0;
    const int32_t* my_rank = rank_tab + (row_ok ? my_row : 0) * n_ch;
    for (;;) {
        if (tid == 0) s_row = atomicAdd(&g_queue[slot][0], 1u);
        __syncthreads();
        const unsigned int ticket = s_row;
        if (ticket >= (unsigned int)n_geo) break;
        const int r = n_geo - 1 - (int)ticket;                 // the long rows sit at the high cell indices: they go first
        const int grp = geo_row_ptr[r], cnt = geo_row_ptr[r + 1] - grp;
        double c[4][2] = {};                                   // D[row oct][vectors 2 quad, 2 quad + 1]: four independent chains of MMAs
        if (cnt > 0 && first_gamma >= 0) {
            const int32_t* cfirst = col_idx + (chan_off[first_gamma] * nnz_geo + (int64_t)ncoupled[first_gamma] * grp);
            const double* vrow = values + (my_off + (int64_t)my_nc * grp);          // this lane's CSR row (gamma, r)
            const int S = min(cnt, cap);
            for (int s0 = 0; s0 < cnt; s0 += S) {
                const int cs = min(S, cnt - s0);
                const int gpc = max(1, cap / cs);              // channels per chunk
                __syncthreads();
                for (int s = tid; s < cs; s += GM_THREADS) gcol[s] = __ldg(cfirst + s0 + s) - first_gp * n_geo;
                for (int glo = 0; glo < n_ch; glo += gpc) {
                    const int ghi = min(n_ch, glo + gpc);
                    __syncthreads();                           // gcol is there; the previous X tile is no longer read
                    // x comes interleaved (xi[column][8]): a thread takes tile entries i = tid, tid + GM_THREADS, ... and moves the
                    // 64 bytes of each as four 16-byte loads; (channel gg, geometric entry s) of i advance without divisions
                    {
                        const int n_tile = (ghi - glo) * cs;
                        const int dq = GM_THREADS / cs, dr = GM_THREADS - dq * cs;
                        int gg = tid / cs, s = tid - gg * cs;
                        for (int i = tid; i < n_tile; i += GM_THREADS) {
                            const double2* xp = reinterpret_cast<const double2*>(xi + ((int64_t)(glo + gg) * n_geo + gcol[s]) * 8);
                            const double2 x0 = __ldg(xp), x1 = __ldg(xp + 1), x2 = __ldg(xp + 2), x3 = __ldg(xp + 3);
                            double* d = X + i;
                            d[0] = x0.x; d[ps] = x0.y; d[2 * ps] = x1.x; d[3 * ps] = x1.y;
                            d[4 * ps] = x2.x; d[5 * ps] = x2.y; d[6 * ps] = x3.x; d[7 * ps] = x3.y;
                            gg += dq; s += dr;
                            if (s >= cs) { s -= cs; ++gg; }
                        }
                    }
                    __syncthreads();
                    // this warp's share of the chunk's channels gamma', two at a time (their value loads are independent);
                    // per gamma' the cs tile entries in steps of 4 (one MMA each), GM_UNR steps of loads in flight together
                    for (int gp = glo + (grp_id < n_grp ? wig : n_ch); gp < ghi; gp += 2 * wpg) {
                        const int gq = gp + wpg;
                        const bool has_q = gq < ghi;
                        const int rk = row_ok ? my_rank[gp] : -1;                        // rank of gamma' in this lane's row, or -1
                        const int rq = (row_ok && has_q) ? my_rank[gq] : -1;
                        const double* vp = vrow + ((int64_t)max(rk, 0) * cnt + s0 + quad);
                        const double* vq = vrow + ((int64_t)max(rq, 0) * cnt + s0 + quad);
                        const double* xb = X + oct * ps + (gp - glo) * cs + quad;        // B fragment: plane (vector) oct, entry s + quad
                        const double* xq = xb + wpg * cs;
                        for (int s = 0; s < cs; s += 4 * GM_UNR) {
                            double a[GM_UNR], aq[GM_UNR];
#pragma unroll
                            for (int k = 0; k < GM_UNR; ++k) {
                                const bool in = s + 4 * k + quad < cs;
                                a[k] = (in && rk >= 0) ? ld_value_l2_256(vp + s + 4 * k) : 0.0;
                                aq[k] = (in && rq >= 0) ? ld_value_l2_256(vq + s + 4 * k) : 0.0;
                            }
#pragma unroll
                            for (int k = 0; k < GM_UNR; ++k) {
                                if (s + 4 * k >= cs) break;                               // warp-uniform
                                const bool in = s + 4 * k + quad < cs;
                                dmma_884g(c[k & 1][0], c[k & 1][1], a[k], in ? xb[s + 4 * k] : 0.0);
                                if (has_q) dmma_884g(c[2 + (k & 1)][0], c[2 + (k & 1)][1], aq[k], in ? xq[s + 4 * k] : 0.0);
                            }
                        }
                    }
                }
            }
        }
        // ---- the partial sums of the wpg warps of a row group, added in a fixed order
        *reinterpret_cast<double2*>(ypart + (size_t)warp * 64 + oct * 8 + 2 * quad) =
            make_double2((c[0][0] + c[1][0]) + (c[2][0] + c[3][0]), (c[0][1] + c[1][1]) + (c[2][1] + c[3][1]));
        __syncthreads();
        for (int i = tid; i < n_ch * 8; i += GM_THREADS) {
            const int ga = i >> 3, v = i & 7;
            const double* pp = ypart + (size_t)((ga >> 3) * wpg) * 64 + (ga & 7) * 8 + v;
            double sum = 0.0;
            for (int w = 0; w < wpg; ++w) sum += pp[w * 64];
            if (v < nv) y[v * ldx + (int64_t)ga * n_geo + r] = sum;
        }
    }
    // the last CTA of the launch puts the queue slot back to zero
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(&g_queue[slot][1], 1u) == gridDim.x - 1) {
            g_queue[slot][0] = 0u;
            g_queue[slot][1] = 0u;
            __threadfence();
        }
    }
}

}  // namespace

// Scratch of wpcd_perm_apply_blocked_noalloc: the interleaved copy of up to 8 x vectors of a matrix with at most
// WPCD_NOALLOC_MAX_ROWS rows (16 MiB), held by every device that loads the library until the process exits.  In host code this
// name is a host-side stand-in, not a device address: the launcher below asks cudaGetSymbolAddress for the address.
static __device__ __align__(256) double g_noalloc_xi[(size_t)WPCD_NOALLOC_MAX_ROWS * 8];

namespace wpcd_detail {

bool use_pdl();

// One vector: 256 threads and an x tile of 1536 doubles (measured on a B200, N = 150, 26 - 62 channels: 1280 - 1792
// doubles stream the values at the HBM copy rate; from 2048 on fewer CTAs fit an SM and the rate drops by a quarter).
// Several vectors: the tile holds NV planes; it is kept large enough for a whole average geometric row (3072 doubles
// per vector), because every (channel chunk, row) costs a warp reduction per vector, and the CTA grows to 512 / 1024
// threads so that the SM still has 32 - 64 warps streaming.
template <int NV, int THREADS>
static cudaError_t launch_georow(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr, const int32_t* col_idx,
                                 const double* values, const double* x, double* y, int64_t ldx, cudaStream_t st)
{
    static std::atomic<unsigned int> next_slot{0};
    const int n_geo = g->n_p * g->n_q;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int forced = g_debug.blocked_tile_doubles.load();
    const int cap = forced > 0 ? forced : (NV == 1 ? 1536 : 3072);        // doubles per vector
    const size_t smem = sizeof(double) * ((size_t)cap * NV + (size_t)ch->n_ch * NV) + sizeof(int32_t) * (size_t)cap;
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    cudaError_t err = raise_dyn_smem(spmv_georow_kernel<NV, THREADS>, smem);
    if (err != cudaSuccess) return err;
    int per_sm = 0;
    err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spmv_georow_kernel<NV, THREADS>, THREADS, smem);
    if (err != cudaSuccess) return err;
    const int blocks = std::max(1, std::min(n_geo, sms * std::max(1, per_sm)));
    const int slot = (int)(next_slot.fetch_add(1) % GB_RING);
    ++g_launches;
    spmv_georow_kernel<NV, THREADS><<<blocks, THREADS, smem, st>>>(n_geo, ch->n_ch, geo_row_ptr, col_idx, values, ch->chan_off_dev,
                                                                  ch->ncoupled_dev, ch->run_ptr_dev, ch->runs_dev, ch->first_gamma, ch->first_gp,
                                                                  x, y, ldx, cap, slot);
    return cudaGetLastError();
}

// nv <= 8 vectors on the tensor cores (n_ch <= 64): tile of 2560 doubles per vector, one 512-thread CTA per SM.  The planes
// of the vectors nv .. 7 are zero and their results are not written.
static cudaError_t launch_georow_mma8(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr, const int32_t* col_idx,
                                      const double* values, const double* x, double* y, int64_t ldx, int nv, cudaStream_t st)
{
    static std::atomic<unsigned int> next_slot{1u << 20};
    const int n_geo = g->n_p * g->n_q;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int forced = g_debug.blocked_tile_doubles.load();
    const int cap = forced > 0 ? forced : 2560;
    const size_t smem = sizeof(double) * ((size_t)(cap + 4) * 8 + (size_t)GM_WARPS * 64) + sizeof(int32_t) * ((size_t)cap + (size_t)ch->n_ch * ch->n_ch);
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    cudaError_t err = raise_dyn_smem(spmv_georow_mma8_kernel, smem);
    if (err != cudaSuccess) return err;
    const int blocks = std::max(1, std::min(n_geo, sms));
    const int slot = (int)(next_slot.fetch_add(1) % GB_RING);
    // scratch for the interleaved copy of the 8 vectors: stream-ordered allocation, released behind the product
    const int64_t rows = (int64_t)ch->n_ch * n_geo;
    double* xi = nullptr;
    err = cudaMallocAsync(reinterpret_cast<void**>(&xi), sizeof(double) * 8 * (size_t)rows, st);
    if (err != cudaSuccess) return err;
    g_launches += 2;
    interleave8_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, st>>>(rows, nv, x, ldx, xi);
    spmv_georow_mma8_kernel<<<blocks, GM_THREADS, smem, st>>>(n_geo, ch->n_ch, geo_row_ptr, col_idx, values, ch->chan_off_dev, ch->ncoupled_dev,
                                                             ch->run_ptr_dev, ch->runs_dev, ch->first_gamma, ch->first_gp, xi, y, ldx, nv, cap, slot);
    err = cudaGetLastError();
    const cudaError_t ferr = cudaFreeAsync(xi, st);
    return err != cudaSuccess ? err : ferr;
}

cudaError_t launch_spmv_blocked(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr, const int32_t* col_idx,
                                const double* values, const double* x, double* y, int n_vec, cudaStream_t st)
{
    const int64_t rows = (int64_t)ch->n_ch * g->n_p * g->n_q;
    int v = 0;
    while (v < n_vec) {
        const double* xv = x + (int64_t)v * rows;
        double* yv = y + (int64_t)v * rows;
        cudaError_t err;
        // 3 .. 8 vectors: one tensor-core pass (6.7 ms on the 3.2e9-nonzero matrix whatever their number; the scalar kernels
        // take 6.8 ms for 4 vectors, 4.4 for 2, 3.9 for 1)
        if (n_vec - v >= 3 && ch->n_ch <= 8 * GM_GROUPS && g_debug.blocked_no_mma.load() == 0) {
            const int nv = std::min(8, n_vec - v);
            err = launch_georow_mma8(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, nv, st);
            v += nv;
        }
        else if (n_vec - v >= 8) { err = launch_georow<8, 1024>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 8; }
        else if (n_vec - v >= 4) { err = launch_georow<4, 1024>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 4; }
        else if (n_vec - v >= 2) { err = launch_georow<2, 512>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 2; }
        else { err = launch_georow<1, 256>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 1; }
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

// The tensor-core pass with its scratch in g_noalloc_xi: no cudaMalloc / cudaFree of any kind.  nv = 1 .. 8 vectors, n_ch <= 64,
// rows <= WPCD_NOALLOC_MAX_ROWS (checked by the caller).  Every call uses the same array: the interleave kernel rewrites all
// 8 rows words the product reads (zeros for the vectors nv .. 7), so nothing of an earlier call is seen; two calls that
// overlap on the GPU (different streams) race on it.
cudaError_t launch_spmv_blocked_noalloc(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr, const int32_t* col_idx,
                                        const double* values, const double* x, double* y, int nv, cudaStream_t st)
{
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static double* xi_of_device[MAX_DEV] = {};             // device address of g_noalloc_xi, per device
    static std::atomic<unsigned int> next_slot{1u << 21};
    int dev = 0, sms = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
    double* xi = nullptr;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (!xi_of_device[dev]) {                          // once per device, with that device current
            void* ptr = nullptr;
            err = cudaGetSymbolAddress(&ptr, g_noalloc_xi);
            if (err != cudaSuccess) return err;
            xi_of_device[dev] = static_cast<double*>(ptr);
        }
        xi = xi_of_device[dev];
    }
    err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (err != cudaSuccess) return err;
    const int n_geo = g->n_p * g->n_q;
    const int64_t rows = (int64_t)ch->n_ch * n_geo;
    if (rows > WPCD_NOALLOC_MAX_ROWS || ch->n_ch > 8 * GM_GROUPS || nv < 1 || nv > 8) return cudaErrorInvalidValue;
    const int cap = 2560;
    const size_t smem = sizeof(double) * ((size_t)(cap + 4) * 8 + (size_t)GM_WARPS * 64) + sizeof(int32_t) * ((size_t)cap + (size_t)ch->n_ch * ch->n_ch);
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    err = raise_dyn_smem(spmv_georow_mma8_kernel, smem);
    if (err != cudaSuccess) return err;
    const int blocks = std::max(1, std::min(n_geo, sms));
    const int slot = (int)(next_slot.fetch_add(1) % GB_RING);
    g_launches += 2;
    interleave8_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, st>>>(rows, nv, x, rows, xi);
    spmv_georow_mma8_kernel<<<blocks, GM_THREADS, smem, st>>>(n_geo, ch->n_ch, geo_row_ptr, col_idx, values, ch->chan_off_dev, ch->ncoupled_dev,
                                                             ch->run_ptr_dev, ch->runs_dev, ch->first_gamma, ch->first_gp, xi, y, rows, nv, cap, slot);
    return cudaGetLastError();
}

}  // namespace wpcd_detail
