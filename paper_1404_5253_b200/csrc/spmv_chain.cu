// spmv_chain.cu -- y_k = P0 y_{k-1}, k = 1 .. n_iter, y_0 = x: the dependent products of the simple iteration of
// eq. (12) (paper step 5; terms of the Neumann series summed by Pade approximants) for a
// matrix small enough to live on chip.
// ONE cooperative launch does the whole chain: every CTA (one per SM) keeps its slice of rows -- column indices,
// values and row offsets -- in shared memory for all n_iter products, gathers x through L2 (ld.global.cg: the
// previous iterate was written by other SMs), and a grid-wide barrier (release-add / acquire-poll on one counter)
// separates the products.  Rows are split among the CTAs by nonzero count (binary search of row_ptr for the CTA's
// quantiles).
// Measured on a B200 (s-wave lattices, 50 products, per product; ordinary products replayed from a CUDA graph):
//   nnz 6.8e3: 2.14 us here / 1.87 us ordinary;  4.4e4: 2.31 / 2.78;  2.9e5: 4.59 / 4.43;  7.3e5: 7.7 / 7.0.
// The grid barrier costs ~2 us (store ack + release + one poll round trip through L2), as much as a kernel boundary
// under programmatic dependent launch, so the fused chain pays only in a window of sizes; outside it (and for any
// matrix that does not fit) the chain is n_iter ordinary products (spmv.cu).  A variant without barrier (each
// iterate's 8-byte words doubling as ready flags, polled by the gathers) measured slower still (3.5 - 6.5 us).
#include <stdlib.h>

#include <algorithm>
#include <map>
#include <mutex>

#include "wpcd_internal.h"

namespace {

constexpr int CH_TPB = 1024;
constexpr int CH_UNR = 4;

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void red_release_add_u32(unsigned* p, unsigned v)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// all CTAs of the (co-resident, cooperative) grid have finished product k when the counter reaches target
__device__ __forceinline__ void grid_barrier(unsigned* counter, unsigned target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        // release is cumulative over the CTA's stores ordered before it by the barrier above; acquire + the barrier
        // below order every later load of the CTA after the other CTAs' stores (the gathers bypass L1: ld.global.cg)
        red_release_add_u32(counter, 1u);
        while (ld_acquire_u32(counter) < target) {}
    }
    __syncthreads();
}

// CH_UNR gathers of the previous iterate, all issued before the first use
template <typename Index>
__device__ __forceinline__ void gather_iterate(const double* xin, const bool (&in)[CH_UNR], const Index (&c)[CH_UNR],
                                               double (&xv)[CH_UNR])
{
#pragma unroll
    for (int u = 0; u < CH_UNR; ++u) xv[u] = in[u] ? __ldcg(xin + c[u]) : 0.0;
}

constexpr unsigned CH_NO_SLOT = 0xffffffffu;

// Lane slots: row r of the CTA's slice gets L_r = ceil(len_r / CH_UNR) lanes (1 .. 32, never straddling a warp), so a
// row of up to 128 entries is gathered in ONE batch whatever its length, and the CTA's whole slice in
// ceil(slots / 1024) passes: the time of a product is one L2 round trip plus the barrier, not a function of the
// longest row.  A slot descriptor packs (row : 16, lane-in-row : 8, lanes : 8).
__global__ void __launch_bounds__(CH_TPB, 1)
spmv_chain_kernel(int64_t rows, const int64_t* __restrict__ row_ptr, const int32_t* __restrict__ col_idx,
                  const double* __restrict__ values, const double* x, double* y, int n_iter, unsigned* counter,
                  int cap_entries, int cap_rows, int cap_slots)
{
    extern __shared__ __align__(16) unsigned char smem[];
    double* s_val = reinterpret_cast<double*>(smem);                       // [cap_entries]
    int* s_col = reinterpret_cast<int*>(smem + (size_t)8 * cap_entries);   // [cap_entries]
    int* s_rp = s_col + cap_entries;                                       // [cap_rows + 1], relative to e_lo
    unsigned* s_desc = reinterpret_cast<unsigned*>(s_rp + cap_rows + 1);   // [cap_slots]
    int* s_first = reinterpret_cast<int*>(s_desc + cap_slots);             // [cap_rows] first slot of a row
    __shared__ int64_t s_bounds[2];
    __shared__ int s_total;
    const int G = gridDim.x, b = blockIdx.x, tid = threadIdx.x;
    const int64_t nnz = row_ptr[rows];
    if (tid < 2) {
        // rows [r(b), r(b+1)) with r(q) = first row whose row_ptr reaches the q-th nonzero quantile
        const int q = b + tid;
        int64_t r;
        if (q == 0) r = 0;
        else if (q == G) r = rows;
        else {
            const int64_t target = nnz / G * q + (nnz % G) * q / G;
            int64_t lo = 0, hi = rows;
            while (lo < hi) {
                const int64_t mid = (lo + hi) >> 1;
                if (row_ptr[mid] < target) lo = mid + 1; else hi = mid;
            }
            r = lo;
        }
        s_bounds[tid] = r;
    }
    __syncthreads();
    const int64_t r0 = s_bounds[0], r1 = s_bounds[1];
    const int64_t e_lo = row_ptr[r0], e_hi = row_ptr[r1];
    const int64_t nrow64 = r1 - r0;
    const bool fit = (e_hi - e_lo) <= (int64_t)cap_entries && nrow64 <= (int64_t)cap_rows;
    const int nrow = (int)nrow64;
    int total = 0;
    if (fit) {
        for (int64_t e = e_lo + tid; e < e_hi; e += CH_TPB) {
            s_val[e - e_lo] = values[e];
            s_col[e - e_lo] = col_idx[e];
        }
        for (int r = tid; r <= nrow; r += CH_TPB) s_rp[r] = (int)(row_ptr[r0 + r] - e_lo);
        __syncthreads();
        if (tid == 0) {
            int slot = 0;
            for (int r = 0; r < nrow; ++r) {
                const int len = s_rp[r + 1] - s_rp[r];
                int L = (len + CH_UNR - 1) / CH_UNR;
                L = L < 1 ? 1 : (L > 32 ? 32 : L);
                if ((slot & 31) + L > 32) slot = (slot + 31) & ~31;
                s_first[r] = slot;
                slot += L;
            }
            s_total = slot;
        }
        __syncthreads();
        total = s_total;
        if (total <= cap_slots) {
            for (int i = tid; i < total; i += CH_TPB) s_desc[i] = CH_NO_SLOT;
            __syncthreads();
            for (int r = tid; r < nrow; r += CH_TPB) {
                const int len = s_rp[r + 1] - s_rp[r];
                int L = (len + CH_UNR - 1) / CH_UNR;
                L = L < 1 ? 1 : (L > 32 ? 32 : L);
                const int first = s_first[r];
                for (int l = 0; l < L; ++l) s_desc[first + l] = (unsigned)r | ((unsigned)l << 16) | ((unsigned)L << 24);
            }
        }
        __syncthreads();
    }
    const bool slotted = fit && total <= cap_slots;

    const double* xin = x;
    for (int k = 0; k < n_iter; ++k) {
        double* yout = y + (int64_t)k * rows;
        if (slotted) {
            for (int sb = 0; sb < total; sb += CH_TPB) {          // uniform trip count: every lane reaches the shuffles
                const int slot = sb + tid;
                const unsigned desc = slot < total ? s_desc[slot] : CH_NO_SLOT;
                const bool valid = desc != CH_NO_SLOT;
                const int r = (int)(desc & 0xffffu), sub = (int)((desc >> 16) & 0xffu), L = valid ? (int)(desc >> 24) : 1;
                int beg = 0, end = 0;
                if (valid) { beg = s_rp[r]; end = s_rp[r + 1]; }
                double acc = 0.0;
                for (int e0 = beg + sub; e0 < end; e0 += CH_UNR * L) {
                    double a[CH_UNR], xv[CH_UNR];
                    int c[CH_UNR];
                    bool in[CH_UNR];
#pragma unroll
                    for (int u = 0; u < CH_UNR; ++u) {
                        const int e = e0 + u * L;
                        in[u] = e < end;
                        a[u] = in[u] ? s_val[e] : 0.0;
                        c[u] = in[u] ? s_col[e] : 0;
                    }
                    gather_iterate(xin, in, c, xv);
#pragma unroll
                    for (int u = 0; u < CH_UNR; ++u) acc = fma(a[u], xv[u], acc);
                }
                // segmented sum over the L lanes of the row (fixed order: deterministic)
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const double v = __shfl_down_sync(0xffffffffu, acc, o);
                    if (sub + o < L) acc += v;
                }
                if (valid && sub == 0) yout[r0 + r] = acc;
            }
        } else {
            // slice too large for shared memory (one very long row, or far more rows than the average): 8 lanes per
            // row straight from global memory
            constexpr int LPR = 8, NG = CH_TPB / LPR;
            const int grp = tid / LPR, sub = tid % LPR;
            for (int64_t rb = 0; rb < nrow64; rb += NG) {
                const int64_t r = rb + grp;
                const bool valid = r < nrow64;
                int64_t beg = 0, end = 0;
                if (valid) { beg = row_ptr[r0 + r]; end = row_ptr[r0 + r + 1]; }
                double acc = 0.0;
                for (int64_t e0 = beg + sub; e0 < end; e0 += (int64_t)CH_UNR * LPR) {
                    double a[CH_UNR], xv[CH_UNR];
                    int c[CH_UNR];
                    bool in[CH_UNR];
#pragma unroll
                    for (int u = 0; u < CH_UNR; ++u) {
                        const int64_t e = e0 + (int64_t)u * LPR;
                        in[u] = e < end;
                        a[u] = in[u] ? values[e] : 0.0;
                        c[u] = in[u] ? col_idx[e] : 0;
                    }
                    gather_iterate(xin, in, c, xv);
#pragma unroll
                    for (int u = 0; u < CH_UNR; ++u) acc = fma(a[u], xv[u], acc);
                }
#pragma unroll
                for (int o = LPR / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
                if (valid && sub == 0) yout[r0 + r] = acc;
            }
        }
        if (k + 1 < n_iter) grid_barrier(counter, (unsigned)(k + 1) * (unsigned)G);
        xin = yout;
    }
}

struct chain_device {
    int sms = 0, coop = 0, smem_optin = 0;
    unsigned* counters = nullptr;      // ring of barrier counters, one 128-byte line each
    unsigned next = 0;
    int smem_set = 0;                  // dynamic shared memory already granted
};
constexpr int CH_RING = 64;
std::mutex g_chain_mutex;
std::map<int, chain_device> g_chain_dev;

cudaError_t launch_chain(chain_device& d, int64_t rows, const int64_t* row_ptr, const int32_t* col_idx, const double* values,
                         const double* x, double* y, int n_iter, unsigned* counter, int cap_entries, int cap_rows, int cap_slots,
                         size_t smem, cudaStream_t st)
{
    cudaError_t err;
    if ((int)smem > d.smem_set) {
        err = cudaFuncSetAttribute(spmv_chain_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (err != cudaSuccess) return err;
        d.smem_set = (int)smem;
    }
    int per_sm = 0;
    err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, spmv_chain_kernel, CH_TPB, smem);
    if (err != cudaSuccess) return err;
    if (per_sm < 1) return cudaErrorCooperativeLaunchTooLarge;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)d.sms);
    cfg.blockDim = dim3(CH_TPB);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;      // co-residency is checked by the launch: no barrier can hang
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ++wpcd_detail::g_launches;
    return cudaLaunchKernelEx(&cfg, spmv_chain_kernel, rows, row_ptr, col_idx, values, x, y, n_iter, counter, cap_entries,
                              cap_rows, cap_slots);
}

}  // namespace

namespace wpcd_detail {

// *fused = 1 if the chain ran as one cooperative launch, 0 if the matrix does not qualify (the caller then issues
// n_iter ordinary products).
cudaError_t launch_spmv_chain(int64_t rows, const int64_t* row_ptr, const int32_t* col_idx, const double* values,
                              const double* x, double* y, int n_iter, int64_t nnz, cudaStream_t st, int* fused)
{
    *fused = 0;
    const int mode = g_debug.chain_mode.load();
    if (mode == 2 || n_iter < 2 || rows >= (int64_t)1 << 30) return cudaSuccess;
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    std::lock_guard<std::mutex> lock(g_chain_mutex);
    chain_device& d = g_chain_dev[dev];
    if (d.sms == 0) {
        cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&d.coop, cudaDevAttrCooperativeLaunch, dev);
        cudaDeviceGetAttribute(&d.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    }
    if (!d.coop || d.sms <= 0) return cudaSuccess;
    const int64_t smem_budget = (int64_t)d.smem_optin - 2048;
    // per-CTA slice: nnz / G entries (+ one long row of slack) and about rows / G rows; the whole matrix must fit on chip
    const int64_t want_entries = nnz / d.sms + nnz / d.sms / 4 + 2048;
    const int64_t want_rows = std::min<int64_t>(2 * (rows / d.sms) + 256, 65535);
    const int64_t want_slots = want_entries / 2 + want_rows + 64;
    if (want_entries * 12 + (want_rows + 1) * 8 + want_slots * 4 > smem_budget) return cudaSuccess;
    if (mode != 1 && (nnz < 16000 || nnz > 160000)) return cudaSuccess;      // the measured window (file header)
    const int cap_entries = (int)((want_entries + 1) & ~(int64_t)1), cap_rows = (int)want_rows, cap_slots = (int)want_slots;
    const size_t smem = (size_t)cap_entries * 12 + (size_t)(cap_rows + 1) * 8 + (size_t)cap_slots * 4;
    if (!d.counters) {
        err = cudaMalloc(&d.counters, (size_t)CH_RING * 128);
        if (err != cudaSuccess) return err;
    }
    unsigned* counter = d.counters + (size_t)(d.next++ % CH_RING) * 32;
    err = cudaMemsetAsync(counter, 0, sizeof(unsigned), st);
    if (err != cudaSuccess) return err;
    err = launch_chain(d, rows, row_ptr, col_idx, values, x, y, n_iter, counter, cap_entries, cap_rows, cap_slots, smem, st);
    if (err == cudaSuccess) *fused = 1;
    return err;
}

}  // namespace wpcd_detail
