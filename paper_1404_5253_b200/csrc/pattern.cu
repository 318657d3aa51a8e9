// pattern.cu -- "selection of the nonzero elements" (paper step 2).
//
// Compiled with -fmad=false: the structural-nonzero predicate S (R6) is a
// contract of IEEE double +,-,*,/ and comparisons in a fixed expression order, so that
// the CSR pattern is bit-exact against the CPU oracle.
//
// Predicate.  Row cell (i,j): p in [L2,U2], q in [a,b]; column cell (i',j'): p' in [L1,U1],
// q' in [c,d].  From the theta-functions of (A7) with u = q q' x: the cells
// overlap iff the polygon Pi = [a,b]x[c,d] cut by the six half-planes
//   s+t/2 >= L1, |s-t/2| <= U1, s/2+t >= L2, |t-s/2| <= U2        (s = q, t = q')
// has positive area and the energy band L2^2-U1^2 < 3/4 (t^2-s^2) < U2^2-L1^2 meets it.
//
// Work decomposition (B200): one warp per geometric row (i,j).  The six box tests of R6 are
// monotone in j' even in floating point, so for every i' the j' passing all of them form
// one interval found by two binary searches that evaluate THE SAME expressions (N^3 log N
// instead of N^4 tests).  The surviving candidates (~1.3x the nonzeros) are enumerated in
// ascending column order, 32 per step, run through the polygon test, and compacted with
// ballot/popc.
#include <math.h>

#include "wpcd_internal.h"

namespace {

constexpr int WARPS_PER_BLOCK = 8;
constexpr int MAXV = 12;

struct Cell { double a, b, c, d, L1, U1, L2, U2; };

__device__ __forceinline__ double halfplane(int m, double s, double t, const Cell& z)
{
    switch (m) {
    case 0: return (s + 0.5 * t) - z.L1;
    case 1: return z.U1 - (s - 0.5 * t);
    case 2: return z.U1 - (0.5 * t - s);
    case 3: return (0.5 * s + t) - z.L2;
    case 4: return z.U2 - (t - 0.5 * s);
    default: return z.U2 - (0.5 * s - t);
    }
}

// Polygon part of the predicate (the box tests have been applied by the caller).
// Returns 1 for a structural nonzero and then the angular extent of Pi in phi[0..1].
__device__ int overlap_polygon(const Cell& z, double* phi_a, double* phi_b)
{
    double h_lo = z.L2 * z.L2 - z.U1 * z.U1;
    double h_hi = z.U2 * z.U2 - z.L1 * z.L1;
    double ps[2][MAXV], pt[2][MAXV];
    int n = 4, cur = 0;
    ps[0][0] = z.a; pt[0][0] = z.c;
    ps[0][1] = z.b; pt[0][1] = z.c;
    ps[0][2] = z.b; pt[0][2] = z.d;
    ps[0][3] = z.a; pt[0][3] = z.d;
    for (int m = 0; m < 6; ++m) {
        int no = 0, nxt = cur ^ 1;
        double sP = ps[cur][0], tP = pt[cur][0];
        double fP = halfplane(m, sP, tP, z);
        for (int e = 0; e < n; ++e) {
            int e1 = (e + 1 == n) ? 0 : e + 1;
            double sQ = ps[cur][e1], tQ = pt[cur][e1];
            double fQ = halfplane(m, sQ, tQ, z);
            bool inP = fP >= 0.0, inQ = fQ >= 0.0;
            if (inP) { ps[nxt][no] = sP; pt[nxt][no] = tP; ++no; }
            if (inP != inQ) {
                double r = fP / (fP - fQ);
                ps[nxt][no] = sP + (sQ - sP) * r;
                pt[nxt][no] = tP + (tQ - tP) * r;
                ++no;
            }
            sP = sQ; tP = tQ; fP = fQ;
        }
        n = no; cur = nxt;
        if (n < 3) return 0;
    }
    double area2 = 0.0;
    for (int v = 1; v + 1 < n; ++v) {
        double s1 = ps[cur][v] - ps[cur][0], t1 = pt[cur][v] - pt[cur][0];
        double s2 = ps[cur][v + 1] - ps[cur][0], t2 = pt[cur][v + 1] - pt[cur][0];
        area2 = area2 + (s1 * t2 - s2 * t1);
    }
    if (!(area2 > 0.0)) return 0;
    double hmax = 0.75 * (pt[cur][0] * pt[cur][0] - ps[cur][0] * ps[cur][0]), hmin = hmax;
    for (int v = 1; v < n; ++v) {
        double h = 0.75 * (pt[cur][v] * pt[cur][v] - ps[cur][v] * ps[cur][v]);
        hmax = fmax(hmax, h);
        hmin = fmin(hmin, h);
    }
    {
        double s = 4.0 * z.U1 / 3.0, t = 2.0 * z.U1 / 3.0;
        if (s >= z.a && s <= z.b && t >= z.c && t <= z.d && halfplane(0, s, t, z) >= 0.0 && halfplane(2, s, t, z) >= 0.0 &&
            halfplane(3, s, t, z) >= 0.0 && halfplane(4, s, t, z) >= 0.0 && halfplane(5, s, t, z) >= 0.0)
            hmin = fmin(hmin, -(z.U1 * z.U1));
    }
    {
        double s = 2.0 * z.U2 / 3.0, t = 4.0 * z.U2 / 3.0;
        if (s >= z.a && s <= z.b && t >= z.c && t <= z.d && halfplane(0, s, t, z) >= 0.0 && halfplane(1, s, t, z) >= 0.0 &&
            halfplane(2, s, t, z) >= 0.0 && halfplane(3, s, t, z) >= 0.0 && halfplane(5, s, t, z) >= 0.0)
            hmax = fmax(hmax, z.U2 * z.U2);
    }
    if (!(hmax > h_lo)) return 0;
    if (!(hmin < h_hi)) return 0;
    if (phi_a) {
        double lo = 1e300, hi = -1e300;
        for (int v = 0; v < n; ++v) {
            double s = ps[cur][v], t = pt[cur][v];
            if (s == 0.0 && t == 0.0) continue;
            double ang = atan2(t, s);
            lo = fmin(lo, ang);
            hi = fmax(hi, ang);
        }
        *phi_a = lo; *phi_b = hi;
    }
    return 1;
}

// box tests that are monotone non-decreasing in j' (they involve d = q[j'+1] only)
__device__ __forceinline__ bool box_lower(const Cell& z, double d, double h_lo)
{
    return (0.75 * (d * d - z.a * z.a) > h_lo) && (z.b + 0.5 * d > z.L1) && (z.a - 0.5 * d < z.U1) &&
           (0.5 * z.b + d > z.L2) && (0.5 * z.a - d < z.U2);
}
// ... and non-increasing in j' (they involve c = q[j'] only)
__device__ __forceinline__ bool box_upper(const Cell& z, double c, double h_hi)
{
    return (0.75 * (c * c - z.b * z.b) < h_hi) && (0.5 * c - z.b < z.U1) && (c - 0.5 * z.b < z.U2);
}

template <bool WRITE>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32)
geo_pattern_kernel(const double* __restrict__ p, const double* __restrict__ q, int n_p, int n_q,
                   int32_t* __restrict__ geo_counts, const int32_t* __restrict__ geo_row_ptr,
                   int32_t* __restrict__ geo_col, int32_t* __restrict__ geo_row, double2* __restrict__ geo_phi)
{
    extern __shared__ int32_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = blockIdx.x * WARPS_PER_BLOCK + warp;
    if (r >= n_p * n_q) return;
    int32_t* jlo_s = smem + warp * (2 * n_p + 2);   // [n_p]
    int32_t* pre_s = jlo_s + n_p;                    // [n_p+1] exclusive prefix of interval lengths
    const int i = r / n_q, j = r - i * n_q;
    Cell z;
    z.a = q[j]; z.b = q[j + 1]; z.L2 = p[i]; z.U2 = p[i + 1];
    z.c = 0.0; z.d = 0.0; z.L1 = 0.0; z.U1 = 0.0;

    // (1) per i': interval of j' passing the box tests
    int running = 0;
    for (int base = 0; base < n_p; base += 32) {
        int ip = base + lane;
        int len = 0, jlo = 0;
        if (ip < n_p) {
            z.L1 = p[ip]; z.U1 = p[ip + 1];
            double h_lo = z.L2 * z.L2 - z.U1 * z.U1;
            double h_hi = z.U2 * z.U2 - z.L1 * z.L1;
            // first j' with box_lower true
            int lo = 0, hi = n_q;
            while (lo < hi) { int mid = (lo + hi) >> 1; if (box_lower(z, q[mid + 1], h_lo)) hi = mid; else lo = mid + 1; }
            jlo = lo;
            // last j' with box_upper true  (first j' with it false, minus one)
            lo = 0; hi = n_q;
            while (lo < hi) { int mid = (lo + hi) >> 1; if (!box_upper(z, q[mid], h_hi)) hi = mid; else lo = mid + 1; }
            len = lo - jlo; if (len < 0) len = 0;
        }
        // warp exclusive scan of len
        int incl = len;
        for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
        if (ip < n_p) { jlo_s[ip] = jlo; pre_s[ip] = running + incl - len; }
        running += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) pre_s[n_p] = running;
    __syncwarp();
    const int total = running;

    // (2) candidates in ascending column order, polygon test, compaction
    int count = 0;
    const int out_base = WRITE ? geo_row_ptr[r] : 0;
    for (int tb = 0; tb < total; tb += 32) {
        int t = tb + lane;
        int ok = 0, col = 0;
        double pa = 0.0, pb = 0.0;
        if (t < total) {
            int lo = 0, hi = n_p;            // last i' with pre_s[i'] <= t
            while (lo < hi) { int mid = (lo + hi) >> 1; if (pre_s[mid + 1] <= t) lo = mid + 1; else hi = mid; }
            int ip = lo, jp = jlo_s[ip] + (t - pre_s[ip]);
            z.L1 = p[ip]; z.U1 = p[ip + 1]; z.c = q[jp]; z.d = q[jp + 1];
            ok = overlap_polygon(z, WRITE ? &pa : nullptr, &pb);
            col = ip * n_q + jp;
        }
        unsigned m = __ballot_sync(0xffffffffu, ok);
        if (WRITE && ok) {
            int pos = out_base + count + __popc(m & ((1u << lane) - 1u));
            geo_col[pos] = col;
            geo_row[pos] = r;
            geo_phi[pos] = make_double2(pa, pb);
        }
        count += __popc(m);
    }
    if (!WRITE && lane == 0) geo_counts[r] = count;
}

// in place: counts[0..n) -> exclusive prefix, counts[n] = total.  One block.
__global__ void __launch_bounds__(1024) scan_geo_kernel(int32_t* __restrict__ data, int n)
{
    __shared__ int32_t warp_sums[32];
    __shared__ int32_t carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        int idx = base + threadIdx.x;
        int v = idx < n ? data[idx] : 0;
        int incl = v;
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
        if (lane == 31) warp_sums[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int ws = warp_sums[lane], wi = ws;
            for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += u; }
            warp_sums[lane] = wi - ws;
        }
        __syncthreads();
        int carry = carry_s;
        int excl = carry + warp_sums[warp] + incl - v;
        if (idx < n) data[idx] = excl;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) data[n] = carry_s;
}

// row_ptr[(gamma, r)] = chan_off[gamma] * nnz_geo + ncoupled[gamma] * geo_row_ptr[r]
__global__ void rowptr_kernel(const int32_t* __restrict__ geo_row_ptr, int n_geo, int n_ch,
                              const int32_t* __restrict__ ncoupled, const int64_t* __restrict__ chan_off,
                              int64_t* __restrict__ row_ptr)
{
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t rows = (int64_t)n_ch * n_geo;
    if (idx > rows) return;
    int64_t nnz_geo = geo_row_ptr[n_geo];
    if (idx == rows) { row_ptr[idx] = chan_off[n_ch] * nnz_geo; return; }
    int g = (int)(idx / n_geo);
    int r = (int)(idx - (int64_t)g * n_geo);
    row_ptr[idx] = chan_off[g] * nnz_geo + (int64_t)ncoupled[g] * geo_row_ptr[r];
}

}  // namespace

namespace wpcd_detail {

cudaError_t launch_geo_count(const wpcd_grid* g, int32_t* geo_counts_dev, cudaStream_t st)
{
    int n_geo = g->n_p * g->n_q;
    int blocks = (n_geo + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK;
    size_t smem = (size_t)WARPS_PER_BLOCK * (2 * g->n_p + 2) * sizeof(int32_t);
    StageTimer timer(WPCD_STAGE_GEO_COUNT, st);
    geo_pattern_kernel<false><<<blocks, WARPS_PER_BLOCK * 32, smem, st>>>(g->p_dev, g->q_dev, g->n_p, g->n_q, geo_counts_dev,
                                                                          nullptr, nullptr, nullptr, nullptr);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_geo_index(const wpcd_grid* g, const int32_t* geo_row_ptr_dev, int32_t* geo_col, int32_t* geo_row,
                             double2* geo_phi, cudaStream_t st)
{
    int n_geo = g->n_p * g->n_q;
    int blocks = (n_geo + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK;
    size_t smem = (size_t)WARPS_PER_BLOCK * (2 * g->n_p + 2) * sizeof(int32_t);
    StageTimer timer(WPCD_STAGE_GEO_INDEX, st);
    geo_pattern_kernel<true><<<blocks, WARPS_PER_BLOCK * 32, smem, st>>>(g->p_dev, g->q_dev, g->n_p, g->n_q, nullptr,
                                                                         geo_row_ptr_dev, geo_col, geo_row, geo_phi);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_scan_rowptr(const wpcd_grid* g, const wpcd_channels* ch, int32_t* geo_row_ptr_dev, int64_t* row_ptr_dev,
                               cudaStream_t st)
{
    int n_geo = g->n_p * g->n_q;
    StageTimer timer(WPCD_STAGE_SCAN, st);
    scan_geo_kernel<<<1, 1024, 0, st>>>(geo_row_ptr_dev, n_geo);
    ++g_launches;
    int64_t rows = (int64_t)ch->n_ch * n_geo;
    int blocks = (int)((rows + 1 + 255) / 256);
    rowptr_kernel<<<blocks, 256, 0, st>>>(geo_row_ptr_dev, n_geo, ch->n_ch, ch->ncoupled_dev, ch->chan_off_dev, row_ptr_dev);
    ++g_launches;
    return cudaGetLastError();
}

}  // namespace wpcd_detail
