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
                    for (int i = tid; i < (ghi - glo) * cs; i += GB_THREADS) {
                        const int gg = i / cs, s = i - gg * cs;
                        const double* xp = x + (int64_t)(glo + gg) * n_geo + gcol[s];
#pragma unroll
                        for (int v = 0; v < NV; ++v) X[v * cap + i] = __ldg(xp + v * ldx);
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

}  // namespace

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
    cudaError_t err = cudaFuncSetAttribute(spmv_georow_kernel<NV, THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
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

cudaError_t launch_spmv_blocked(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr, const int32_t* col_idx,
                                const double* values, const double* x, double* y, int n_vec, cudaStream_t st)
{
    const int64_t rows = (int64_t)ch->n_ch * g->n_p * g->n_q;
    int v = 0;
    while (v < n_vec) {
        const double* xv = x + (int64_t)v * rows;
        double* yv = y + (int64_t)v * rows;
        cudaError_t err;
        if (n_vec - v >= 8) { err = launch_georow<8, 1024>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 8; }
        else if (n_vec - v >= 4) { err = launch_georow<4, 1024>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 4; }
        else if (n_vec - v >= 2) { err = launch_georow<2, 512>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 2; }
        else { err = launch_georow<1, 256>(g, ch, geo_row_ptr, col_idx, values, xv, yv, rows, st); v += 1; }
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

}  // namespace wpcd_detail
