// wpcd_internal.h -- structures shared by the translation units of libwpcd (product path).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/wpcd.h"

struct wpcd_grid {
    int n_p = 0, n_q = 0;
    std::vector<double> p, q;   // host copies
    char* block_dev = nullptr;  // one device allocation holding p, q, ctrl, stage_off, stage_len
    double* p_dev = nullptr;    // [n_p+1]
    double* q_dev = nullptr;    // [n_q+1]
    // Staged result of the last selection pass on this grid (scratch owned by the handle,
    // written by wpcd_perm_count, consumed by wpcd_perm_build): one slot per box-test candidate.
    int32_t* stage_col = nullptr;       // [stage_cap]  column index, or -1 for a rejected candidate
    double4* stage_ext = nullptr;       // [stage_cap]  vertices of smallest / largest polar angle of Pi (survivors)
    int32_t* stage_off = nullptr;       // [n_p*n_q]    first slot of a geometric row
    int32_t* stage_len = nullptr;       // [n_p*n_q]    number of candidates of a geometric row
    int32_t* ctrl = nullptr;            // [4] device: slot cursor, overflow flag, nnz_geo
    int32_t* ctrl_pinned = nullptr;     // [4] pinned host copy
    int64_t stage_cap = 0;
    bool stage_valid = false;
    bool select_ready = false;          // kernel attributes set
    int64_t stage_nnz_geo = 0;
};

// monomial mu = (k, A, l, l'):  P_k(x) cos^{A+1} sin^{l+l'-A+1} / (zeta1^{l'+1} zeta2^{l+1})
struct wpcd_monomial { int16_t k, A, l, lp; };

struct wpcd_channels {
    int model = 0;
    int n_ch = 0, n_pairs = 0;
    int64_t n_terms = 0;
    bool swave_single = false;   // one channel, one term k=l1=l1'=0, l=l'=0
    double g0 = 0.0;
    std::vector<int32_t> qn;     // [n_ch*6]
    std::vector<int32_t> channel_l;
    std::vector<int32_t> pair_gamma, pair_gammap, term_k, term_l1, term_l1p;
    std::vector<int64_t> term_ptr;
    std::vector<double> term_g;
    // merged monomial form used by the fill kernels
    int n_mu = 0, k_max = 0, l_max = 0;
    std::vector<wpcd_monomial> mu;            // [n_mu]
    std::vector<int32_t> mterm_ptr;           // [n_pairs+1]
    std::vector<int32_t> mterm_mu;            // merged terms: monomial index
    std::vector<double> mterm_g;              //               coefficient
    // device tables
    int32_t* ncoupled_dev = nullptr;          // [n_ch]   number of gamma' coupled to gamma
    int64_t* chan_off_dev = nullptr;          // [n_ch+1] prefix of ncoupled
    int32_t* pair_gamma_dev = nullptr;        // [n_pairs]
    int32_t* pair_gammap_dev = nullptr;       // [n_pairs]
    int32_t* pair_ci_dev = nullptr;           // [n_pairs] rank of gamma' among the coupled of gamma
    wpcd_monomial* mu_dev = nullptr;          // [n_mu]
    int32_t* mterm_ptr_dev = nullptr;         // [n_pairs+1]
    int32_t* mterm_mu_dev = nullptr;
    double* mterm_g_dev = nullptr;
    std::vector<int32_t> ncoupled;
    int64_t total_coupled = 0;
};

namespace wpcd_detail {

void set_error(const std::string& msg);
extern int64_t g_launches;

// RAII stage timer (wpcd_trace_enable): records an event pair around a kernel launch.
struct StageTimer {
    StageTimer(int stage, cudaStream_t st);
    ~StageTimer();
    int stage; cudaStream_t st; cudaEvent_t e0 = nullptr, e1 = nullptr;
};

// Small process-wide cache of device / pinned buffers used for the scratch inside the handles, so
// that creating and destroying handles in a loop does not pay cudaMalloc / cudaFree every time.
void* pool_alloc(size_t bytes, bool pinned, cudaError_t* err);
void pool_free(void* ptr);

// workspace layout for nnz_geo geometric entries (all 256-byte aligned)
struct Workspace {
    int32_t* geo_col;    // [nnz_geo]
    int32_t* geo_row;    // [nnz_geo]
    double2* geo_phi;    // [nnz_geo]  (phi_a, phi_b)
    double* moments;     // [chunk * n_mu] (coupled channels only)
    int64_t chunk;       // geometric elements per moment chunk
    size_t bytes;
};
Workspace carve_workspace(const wpcd_channels* ch, int64_t nnz_geo, void* base);

// pattern.cu  (compiled with -fmad=false: the predicate is an IEEE contract)
cudaError_t ensure_stage(wpcd_grid* g, int64_t want_cap);
cudaError_t launch_geo_select(wpcd_grid* g, int32_t* geo_row_ptr_dev /* out: ptr */, cudaStream_t st);
cudaError_t launch_rowptr(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr_dev, int64_t* row_ptr_dev,
                          cudaStream_t st);
cudaError_t launch_geo_gather(const wpcd_grid* g, const int32_t* geo_row_ptr_dev, int32_t* geo_col, int32_t* geo_row,
                              double2* geo_phi, cudaStream_t st);

// fill.cu
cudaError_t launch_fill_swave(const wpcd_grid* g, const wpcd_channels* ch, int n_quad, const double* xi, const double* w,
                              int64_t nnz_geo, const Workspace& ws, int32_t* col_idx, double* values, cudaStream_t st);
cudaError_t launch_fill_coupled(const wpcd_grid* g, const wpcd_channels* ch, int n_quad, const double* xi, const double* w,
                                int64_t nnz_geo, const Workspace& ws, const int64_t* row_ptr, const int32_t* geo_row_ptr,
                                int32_t* col_idx, double* values, cudaStream_t st);

// spmv.cu
cudaError_t launch_spmv(int64_t rows, const int64_t* row_ptr, const int32_t* col_idx, const double* values,
                        const double* x, double* y, int n_vec, double mean_row, cudaStream_t st);
cudaError_t run_fp64_peak(cudaStream_t st, double* flops_out);

}  // namespace wpcd_detail
