// kernel_apply.cu -- next row of SURVEY.md section 8(f): the Faddeev kernel applied in factored form.
// In the scattering-wave-packet basis the permutation matrix is P = O P0 O^T (eq. 10, PAPER.md:142-144,
// O^l_{ki} of eq. 8) and the kernel of eq. (12) is K = P V1 G1, kept as a
// product of "a very sparse matrix P0, a diagonal matrix G1 and two block matrices":
//     y = O ( P0 ( O^T ( V1 ( G1 .* x ) ) ) ),   x, y complex (interleaved re, im).
// O and V1 act on the pair index (i or k) inside one channel and one q-bin: for every channel gamma,
// Y_gamma = A_gamma X_gamma with X_gamma the n_p x n_q block of the vector -- a batch of small dense
// products, done here on the FP64 tensor cores (mma.sync m8n8k4).  A complex vector is the real
// n_p x (2 n_q) block with interleaved columns, because A is real.
#include "wpcd_internal.h"

namespace {

constexpr int BT = 32;        // tile edge
constexpr int BS = 36;        // shared-memory row stride (doubles), = 4 mod 16: conflict-free fragment loads

__device__ __forceinline__ void dmma_884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Y[g][k][c] = sum_i A[g][k][i] X[g][i][c]   (TRANS: A[g][i][k]);  X, Y: [n_ch][n_p][n_cols] row-major.
// grid = (ceil(n_cols/32), ceil(n_p/32), n_ch), 128 threads: warp w owns rows 8w..8w+7 of the 32 x 32 tile.
template <bool TRANS>
__global__ void __launch_bounds__(128)
block_apply_kernel(int n_p, int n_cols, const double* __restrict__ A, const double* __restrict__ X, double* __restrict__ Y)
{
    __shared__ double As[BT * BS];   // As[k][i]
    __shared__ double Xs[BT * BS];   // Xs[i][c]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int c0 = blockIdx.x * BT, k0 = blockIdx.y * BT;
    const size_t g = blockIdx.z;
    const double* Ag = A + g * (size_t)n_p * n_p;
    const double* Xg = X + g * (size_t)n_p * n_cols;
    double* Yg = Y + g * (size_t)n_p * n_cols;
    double acc0[4], acc1[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { acc0[j] = 0.0; acc1[j] = 0.0; }
    for (int i0 = 0; i0 < n_p; i0 += BT) {
        for (int t = threadIdx.x; t < BT * BT; t += 128) {
            const int r = t >> 5, c = t & 31;
            // A tile: element (k0 + r, i0 + c); zero outside the matrix
            double a = 0.0;
            if (k0 + r < n_p && i0 + c < n_p) a = TRANS ? Ag[(size_t)(i0 + c) * n_p + k0 + r] : Ag[(size_t)(k0 + r) * n_p + i0 + c];
            As[r * BS + c] = a;
            double xv = 0.0;
            if (i0 + r < n_p && c0 + c < n_cols) xv = Xg[(size_t)(i0 + r) * n_cols + c0 + c];
            Xs[r * BS + c] = xv;
        }
        __syncthreads();
#pragma unroll
        for (int kt = 0; kt < BT / 4; ++kt) {
            const double a = As[(8 * warp + (lane >> 2)) * BS + 4 * kt + (lane & 3)];
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma_884(acc0[j], acc1[j], a, Xs[(4 * kt + (lane & 3)) * BS + 8 * j + (lane >> 2)]);
        }
        __syncthreads();
    }
    const int k = k0 + 8 * warp + (lane >> 2);
    if (k < n_p) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = c0 + 8 * j + 2 * (lane & 3);
            if (c < n_cols) Yg[(size_t)k * n_cols + c] = acc0[j];
            if (c + 1 < n_cols) Yg[(size_t)k * n_cols + c + 1] = acc1[j];
        }
    }
}

// y = g .* x, complex, elementwise (the diagonal channel resolvent G1, eq. 20a/20b are closed forms of ref. [16])
__global__ void __launch_bounds__(256) diag_scale_kernel(int64_t n, const double2* __restrict__ g, const double2* __restrict__ x, double2* __restrict__ y)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const double2 a = g[t], b = x[t];
    y[t] = make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

}  // namespace

namespace wpcd_detail {

cudaError_t launch_block_apply(int n_ch, int n_p, int n_cols, const double* A, bool transpose, const double* X, double* Y, cudaStream_t st)
{
    if (n_ch == 0 || n_p == 0 || n_cols == 0) return cudaSuccess;
    dim3 grid((n_cols + BT - 1) / BT, (n_p + BT - 1) / BT, n_ch);
    if (transpose) block_apply_kernel<true><<<grid, 128, 0, st>>>(n_p, n_cols, A, X, Y);
    else block_apply_kernel<false><<<grid, 128, 0, st>>>(n_p, n_cols, A, X, Y);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_diag_scale(int64_t n, const double* g, const double* x, double* y, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    diag_scale_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, reinterpret_cast<const double2*>(g), reinterpret_cast<const double2*>(x),
                                                                   reinterpret_cast<double2*>(y));
    ++g_launches;
    return cudaGetLastError();
}

}  // namespace wpcd_detail
