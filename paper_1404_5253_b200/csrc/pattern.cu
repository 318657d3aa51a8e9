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
// Work decomposition (B200), ONE evaluation of the predicate per step:
//   geo_select_kernel   a CTA owns ROWS_PER_BLOCK geometric rows.
//     phase 1  (lane = i') the six box tests of R6 are monotone in j' even in floating point,
//              so for every i' the j' passing all of them form one interval.  A guess of its
//              ends comes from closed-form thresholds and two plain binary searches over the
//              q nodes; the ends are then fixed up with THE EXACT box expressions, so the
//              interval is the one an exhaustive scan would give (N^3 log N cheap compares
//              and ~4 N^3 exact box evaluations instead of N^4 tests).
//     phase 2  (thread = candidate, all rows of the CTA pooled for lane balance) the polygon
//              test; the verdict, the column and the angular extent of Pi go to a staging
//              slot that the CTA reserved with one atomicAdd (slots are per candidate, in
//              ascending column order inside a row, so the result does not depend on the
//              order in which CTAs run).
//              The CTA that finishes last scans the per-row survivor counts -> geo_row_ptr.
//   rowptr_kernel       geo_row_ptr x channel coupling -> row_ptr of the full matrix.
//   geo_gather_kernel   (wpcd_perm_build) warp per row: ballot-compaction of the staged
//                       verdicts into the ascending column list geo_col / geo_row / geo_phi.
#include <math.h>

#include <map>
#include <mutex>

#include "wpcd_internal.h"

namespace {

constexpr int TPB = 256;
constexpr int WARPS = TPB / 32;
constexpr int ROWS_PER_BLOCK = 8;
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
// tan1 = (4 U1 / 3, 2 U1 / 3) and tan2 = (2 U2 / 3, 4 U2 / 3) are the tangent points of R6,
// tabulated per bin with exactly these expressions.  Returns 1 for a structural nonzero and then
// the vertices of Pi of smallest and largest polar angle in ext = (s_lo, t_lo, s_hi, t_hi).
__device__ int overlap_polygon(const Cell& z, double2 tan1, double2 tan2, double4* ext)
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
        double s = tan1.x, t = tan1.y;
        if (s >= z.a && s <= z.b && t >= z.c && t <= z.d && halfplane(0, s, t, z) >= 0.0 && halfplane(2, s, t, z) >= 0.0 &&
            halfplane(3, s, t, z) >= 0.0 && halfplane(4, s, t, z) >= 0.0 && halfplane(5, s, t, z) >= 0.0)
            hmin = fmin(hmin, -(z.U1 * z.U1));
    }
    {
        double s = tan2.x, t = tan2.y;
        if (s >= z.a && s <= z.b && t >= z.c && t <= z.d && halfplane(0, s, t, z) >= 0.0 && halfplane(1, s, t, z) >= 0.0 &&
            halfplane(2, s, t, z) >= 0.0 && halfplane(3, s, t, z) >= 0.0 && halfplane(5, s, t, z) >= 0.0)
            hmax = fmax(hmax, z.U2 * z.U2);
    }
    if (!(hmax > h_lo)) return 0;
    if (!(hmin < h_hi)) return 0;
    // Angular extent of Pi (rule R1b of DESIGN.md R7): the vertices of smallest and largest
    // polar angle, found with cross products (all vertices lie in the closed first quadrant).
    // Not part of the bit-exact contract: phi enters the VALUES only.
    double s_lo = 0.0, t_lo = 0.0, s_hi = 0.0, t_hi = 0.0;
    bool have = false;
    for (int v = 0; v < n; ++v) {
        double s = ps[cur][v], t = pt[cur][v];
        if (s == 0.0 && t == 0.0) continue;       // the origin has no angle
        if (!have) { s_lo = s_hi = s; t_lo = t_hi = t; have = true; continue; }
        if (t * s_lo < t_lo * s) { s_lo = s; t_lo = t; }
        if (t * s_hi > t_hi * s) { s_hi = s; t_hi = t; }
    }
    *ext = make_double4(s_lo, t_lo, s_hi, t_hi);
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

// ctrl words (device, owned by the grid handle)
constexpr int CTRL_CURSOR = 0;     // staging slots handed out so far
constexpr int CTRL_OVERFLOW = 1;   // set when the staging capacity was too small
constexpr int CTRL_TICKET = 2;     // CTAs finished (the last one runs the scan)
constexpr int CTRL_RESULT = 4;     // [4] cursor, [5] overflow, [6] nnz_geo of the finished pass (read back by the host)

__global__ void __launch_bounds__(TPB, 4)
geo_select_kernel(const double* __restrict__ p_g, const double* __restrict__ q_g, int n_p, int n_q, int cap,
                  int32_t* __restrict__ geo_counts, int32_t* __restrict__ stage_off, int32_t* __restrict__ stage_len,
                  int32_t* __restrict__ stage_col, double4* __restrict__ stage_ext, int32_t* __restrict__ ctrl)
{
    extern __shared__ __align__(16) double smem_d[];     // 16 bytes: the tangent table is read as double2
    double2* tanp = reinterpret_cast<double2*>(smem_d);          // [n_p] (4 U / 3, 2 U / 3), U = p[i+1]
    double* p = smem_d + 2 * n_p;             // [n_p+1]
    double* q = p + (n_p + 1);                // [n_q+1]
    int32_t* jlo_s = reinterpret_cast<int32_t*>(q + (n_q + 1));   // [ROWS][n_p]
    int32_t* pre_s = jlo_s + ROWS_PER_BLOCK * n_p;                // [ROWS][n_p+1] exclusive prefix of interval lengths
    __shared__ int32_t cbase[ROWS_PER_BLOCK + 1];                  // candidates before row w of this CTA
    __shared__ int32_t rowcnt[ROWS_PER_BLOCK];
    __shared__ int32_t iplo_s[ROWS_PER_BLOCK], iphi_s[ROWS_PER_BLOCK];
    __shared__ int32_t slot_base;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_geo = n_p * n_q;
    const int row0 = blockIdx.x * ROWS_PER_BLOCK;
    for (int t = threadIdx.x; t <= n_p; t += TPB) p[t] = p_g[t];
    for (int t = threadIdx.x; t <= n_q; t += TPB) q[t] = q_g[t];
    for (int t = threadIdx.x; t < n_p; t += TPB) { const double U = p_g[t + 1]; tanp[t] = make_double2(4.0 * U / 3.0, 2.0 * U / 3.0); }
    if (threadIdx.x < ROWS_PER_BLOCK) rowcnt[threadIdx.x] = 0;
    __syncthreads();

    // ---- phase 1: per (row, i') the interval of j' that passes the box tests
    for (int w = warp; w < ROWS_PER_BLOCK; w += WARPS) {
        const int r = row0 + w;
        int32_t* jlo_w = jlo_s + w * n_p;
        int32_t* pre_w = pre_s + w * (n_p + 1);
        int running = 0;
        if (r < n_geo) {
            const int i = r / n_q, j = r - i * n_q;
            Cell z;
            z.a = q[j]; z.b = q[j + 1]; z.L2 = p[i]; z.U2 = p[i + 1];
            z.c = 0.0; z.d = 0.0;
            // i' outside [ip_lo, ip_hi) cannot pass the box tests: they need, for some cell of the q
            // grid, L1 < b + q'/2, L1^2 < U2^2 + 3/4 (b^2 - q'^2), U1 > a - q'/2, U1 > q'/2 - b and
            // U1^2 > L2^2 - 3/4 (q'^2 - a^2).  One bin of slack on each side covers the rounding.
            int ip_lo = 0, ip_hi = n_p;
            {
                const double qmin = q[0], qmax = q[n_q];
                const double eU = z.U2 * z.U2 + 0.75 * (z.b * z.b - qmin * qmin);
                const double PU = eU > 0.0 ? fmin(z.b + 0.5 * qmax, sqrt(eU)) : -1.0;
                const double eL = z.L2 * z.L2 - 0.75 * (qmax * qmax - z.a * z.a);
                double PL = fmax(z.a - 0.5 * qmax, 0.5 * qmin - z.b);
                if (eL > 0.0) PL = fmax(PL, sqrt(eL));
                int lo = 0, hi = n_p;   // first i' with p[i'+1] > PL
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (p[mid + 1] > PL) hi = mid; else lo = mid + 1; }
                ip_lo = lo > 0 ? lo - 1 : 0;
                lo = 0; hi = n_p;       // first i' with p[i'] >= PU
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (p[mid] >= PU) hi = mid; else lo = mid + 1; }
                ip_hi = lo < n_p ? lo + 1 : n_p;
                if (ip_hi < ip_lo) ip_hi = ip_lo;
            }
            if (lane == 0) { iplo_s[w] = ip_lo; iphi_s[w] = ip_hi; pre_w[ip_lo] = 0; }
            for (int base = ip_lo; base < ip_hi; base += 32) {
                const int ip = base + lane;
                int len = 0, jlo = 0;
                if (ip < ip_hi) {
                    z.L1 = p[ip]; z.U1 = p[ip + 1];
                    const double h_lo = z.L2 * z.L2 - z.U1 * z.U1;
                    const double h_hi = z.U2 * z.U2 - z.L1 * z.L1;
                    // guessed thresholds: box_lower <=> d > t_lo, box_upper <=> c < t_hi (up to rounding)
                    const double e_lo = z.a * z.a + h_lo / 0.75;
                    double t_lo = e_lo > 0.0 ? sqrt(e_lo) : -1.0;
                    t_lo = fmax(t_lo, fmax(2.0 * (z.L1 - z.b), 2.0 * (z.a - z.U1)));
                    t_lo = fmax(t_lo, fmax(z.L2 - 0.5 * z.b, 0.5 * z.a - z.U2));
                    const double e_hi = z.b * z.b + h_hi / 0.75;
                    double t_hi = e_hi > 0.0 ? sqrt(e_hi) : -1.0;
                    t_hi = fmin(t_hi, fmin(2.0 * (z.U1 + z.b), z.U2 + 0.5 * z.b));
                    // first j' with q[j'+1] > t_lo
                    int lo = 0, hi = n_q;
                    while (lo < hi) { const int mid = (lo + hi) >> 1; if (q[mid + 1] > t_lo) hi = mid; else lo = mid + 1; }
                    // exact ends: first j' with box_lower true
                    while (lo > 0 && box_lower(z, q[lo], h_lo)) --lo;
                    while (lo < n_q && !box_lower(z, q[lo + 1], h_lo)) ++lo;
                    jlo = lo;
                    // first j' with q[j'] >= t_hi, then exactly: first j' with box_upper false
                    lo = 0; hi = n_q;
                    while (lo < hi) { const int mid = (lo + hi) >> 1; if (q[mid] >= t_hi) hi = mid; else lo = mid + 1; }
                    while (lo > 0 && !box_upper(z, q[lo - 1], h_hi)) --lo;
                    while (lo < n_q && box_upper(z, q[lo], h_hi)) ++lo;
                    len = lo - jlo; if (len < 0) len = 0;
                }
                int incl = len;
                for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
                if (ip < ip_hi) { jlo_w[ip] = jlo; pre_w[ip] = running + incl - len; }
                running += __shfl_sync(0xffffffffu, incl, 31);
            }
            if (lane == 0) pre_w[ip_hi] = running;
        } else if (lane == 0) { iplo_s[w] = 0; iphi_s[w] = 0; }
        if (lane == 0) cbase[w + 1] = running;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int acc = 0;
        cbase[0] = 0;
        for (int w = 0; w < ROWS_PER_BLOCK; ++w) { const int t = cbase[w + 1]; cbase[w + 1] = acc + t; acc += t; }
        int base = acc > 0 ? atomicAdd(&ctrl[CTRL_CURSOR], acc) : 0;
        if (acc > 0 && (base > cap - acc)) { atomicExch(&ctrl[CTRL_OVERFLOW], 1); base = -1; }
        slot_base = base;
    }
    __syncthreads();
    const int total = cbase[ROWS_PER_BLOCK];
    const int sbase = slot_base;

    // ---- phase 2: polygon test of every candidate of the CTA
    for (int cidx = threadIdx.x; cidx < total; cidx += TPB) {
        int w = 0;
#pragma unroll
        for (int s = ROWS_PER_BLOCK / 2; s > 0; s >>= 1) if (cbase[w + s] <= cidx) w += s;
        const int t = cidx - cbase[w];
        const int32_t* pre_w = pre_s + w * (n_p + 1);
        int lo = iplo_s[w], hi = iphi_s[w];   // the i' whose interval holds candidate t
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (pre_w[mid + 1] <= t) lo = mid + 1; else hi = mid; }
        const int ip = lo, jp = jlo_s[w * n_p + ip] + (t - pre_w[ip]);
        const int r = row0 + w;
        const int i = r / n_q, j = r - i * n_q;
        Cell z;
        z.a = q[j]; z.b = q[j + 1]; z.L2 = p[i]; z.U2 = p[i + 1];
        z.L1 = p[ip]; z.U1 = p[ip + 1]; z.c = q[jp]; z.d = q[jp + 1];
        double4 ext;
        const double2 t1 = tanp[ip], t2 = tanp[i];
        const int ok = overlap_polygon(z, t1, make_double2(t2.y, t2.x), &ext);
        if (ok) atomicAdd(&rowcnt[w], 1);
        if (sbase >= 0) {
            stage_col[sbase + cidx] = ok ? ip * n_q + jp : -1;
            if (ok) stage_ext[sbase + cidx] = ext;
        }
    }
    __syncthreads();
    if (threadIdx.x < ROWS_PER_BLOCK && row0 + threadIdx.x < n_geo) {
        const int w = threadIdx.x;
        geo_counts[row0 + w] = rowcnt[w];
        stage_off[row0 + w] = sbase >= 0 ? sbase + cbase[w] : 0;
        stage_len[row0 + w] = sbase >= 0 ? cbase[w + 1] - cbase[w] : 0;
    }

    // ---- a2: the CTA that finishes last turns the counts into geo_row_ptr (in place), publishes
    // (cursor, overflow, nnz_geo) for the host and re-arms the control words for the next pass
    __shared__ int32_t is_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) is_last = atomicAdd(&ctrl[CTRL_TICKET], 1) == (int)gridDim.x - 1;
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    __shared__ int32_t wsum[WARPS];
    const int chunk = (n_geo + TPB - 1) / TPB;
    const int first = threadIdx.x * chunk, last = min(n_geo, first + chunk);
    int sum = 0;
    for (int k = first; k < last; ++k) sum += __ldcg(geo_counts + k);
    int incl = sum;
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    int excl = incl - sum;
    for (int k = 0; k < warp; ++k) excl += wsum[k];
    for (int k = first; k < last; ++k) { const int v = __ldcg(geo_counts + k); geo_counts[k] = excl; excl += v; }
    if (threadIdx.x == TPB - 1) {
        geo_counts[n_geo] = excl;
        ctrl[CTRL_RESULT + 0] = atomicAdd(&ctrl[CTRL_CURSOR], 0);
        ctrl[CTRL_RESULT + 1] = atomicAdd(&ctrl[CTRL_OVERFLOW], 0);
        ctrl[CTRL_RESULT + 2] = excl;
        ctrl[CTRL_CURSOR] = 0; ctrl[CTRL_OVERFLOW] = 0; ctrl[CTRL_TICKET] = 0;
    }
}

// Staged verdicts of one row -> ascending column list.  One warp per geometric row.
__global__ void __launch_bounds__(TPB)
geo_gather_kernel(int n_geo, const int32_t* __restrict__ geo_row_ptr, const int32_t* __restrict__ stage_off,
                  const int32_t* __restrict__ stage_len, const int32_t* __restrict__ stage_col,
                  const double4* __restrict__ stage_ext, int32_t* __restrict__ geo_col, int32_t* __restrict__ geo_row,
                  double2* __restrict__ geo_phi)
{
    const int lane = threadIdx.x & 31;
    const int r = blockIdx.x * WARPS + (threadIdx.x >> 5);
    if (r >= n_geo) return;
    const int off = stage_off[r], len = stage_len[r];
    int out = geo_row_ptr[r];
    for (int tb = 0; tb < len; tb += 32) {
        const int t = tb + lane;
        const int col = t < len ? stage_col[off + t] : -1;
        const unsigned m = __ballot_sync(0xffffffffu, col >= 0);
        if (col >= 0) {
            const int pos = out + __popc(m & ((1u << lane) - 1u));
            geo_col[pos] = col;
            geo_row[pos] = r;
            const double4 ext = stage_ext[off + t];
            geo_phi[pos] = make_double2(atan2(ext.y, ext.x), atan2(ext.w, ext.z));
        }
        out += __popc(m);
    }
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

static size_t select_smem(const wpcd_grid* g)
{
    return sizeof(double) * (size_t)(g->n_p + g->n_q + 2 + 2 * g->n_p) + sizeof(int32_t) * (size_t)ROWS_PER_BLOCK * (2 * g->n_p + 1);
}

cudaError_t ensure_stage(const wpcd_grid* g, int64_t want_cap)
{
    cudaError_t err = cudaSuccess;
    if (!g->select_ready) {
        // the attribute belongs to the kernel (per device), not to the grid, and a call replaces it: keep the largest request
        static std::mutex attr_mutex;
        static std::map<int, size_t> attr_max;
        const size_t need = select_smem(g);
        if (need > 227 * 1024) return cudaErrorInvalidValue;   // n_p beyond what one CTA can stage
        int dev = 0;
        cudaGetDevice(&dev);
        std::lock_guard<std::mutex> lock(attr_mutex);
        size_t& have = attr_max[dev];
        if (need > 32 * 1024 && need > have) {      // the default 48 KB limit counts the static shared memory too
            if ((err = cudaFuncSetAttribute(geo_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need)) != cudaSuccess) return err;
            have = need;
        }
        g->select_ready = true;
    }
    if (want_cap > g->stage_cap) {
        if (want_cap > (int64_t)INT32_MAX) return cudaErrorInvalidValue;
        g->stage_valid = false;
        pool_free(g->stage_col); pool_free(g->stage_ext);
        g->stage_col = nullptr; g->stage_ext = nullptr; g->stage_cap = 0;
        g->stage_col = static_cast<int32_t*>(pool_alloc(sizeof(int32_t) * (size_t)want_cap, false, &err));
        if (err != cudaSuccess) return err;
        g->stage_ext = static_cast<double4*>(pool_alloc(sizeof(double4) * (size_t)want_cap, false, &err));
        if (err != cudaSuccess) return err;
        g->stage_cap = want_cap;
    }
    return cudaSuccess;
}

// Predicate + per-row counts + staged verdicts (a1) and, in its last CTA, the scan (a2).  No sync.
cudaError_t launch_geo_select(const wpcd_grid* g, int32_t* geo_row_ptr_dev, cudaStream_t st)
{
    const int n_geo = g->n_p * g->n_q;
    const int blocks = (n_geo + ROWS_PER_BLOCK - 1) / ROWS_PER_BLOCK;
    StageTimer timer(WPCD_STAGE_GEO_COUNT, st);
    geo_select_kernel<<<blocks, TPB, select_smem(g), st>>>(g->p_dev, g->q_dev, g->n_p, g->n_q, (int)g->stage_cap, geo_row_ptr_dev,
                                                          g->stage_off, g->stage_len, g->stage_col, g->stage_ext, g->ctrl);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_rowptr(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr_dev, int64_t* row_ptr_dev,
                          cudaStream_t st)
{
    const int n_geo = g->n_p * g->n_q;
    StageTimer timer(WPCD_STAGE_SCAN, st);
    int64_t rows = (int64_t)ch->n_ch * n_geo;
    int blocks = (int)((rows + 1 + 255) / 256);
    rowptr_kernel<<<blocks, 256, 0, st>>>(geo_row_ptr_dev, n_geo, ch->n_ch, ch->ncoupled_dev, ch->chan_off_dev, row_ptr_dev);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_geo_gather(const wpcd_grid* g, const int32_t* geo_row_ptr_dev, int32_t* geo_col, int32_t* geo_row,
                              double2* geo_phi, cudaStream_t st)
{
    const int n_geo = g->n_p * g->n_q;
    const int blocks = (n_geo + WARPS - 1) / WARPS;
    StageTimer timer(WPCD_STAGE_GEO_INDEX, st);
    geo_gather_kernel<<<blocks, TPB, 0, st>>>(n_geo, geo_row_ptr_dev, g->stage_off, g->stage_len, g->stage_col, g->stage_ext,
                                              geo_col, geo_row, geo_phi);
    ++g_launches;
    return cudaGetLastError();
}

}  // namespace wpcd_detail
