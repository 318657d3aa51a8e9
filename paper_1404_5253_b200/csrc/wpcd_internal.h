// wpcd_internal.h -- structures shared by the translation units of libwpcd (product path).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "../../include/wpcd.h"

struct wpcd_grid {
    int n_p = 0, n_q = 0;
    std::vector<double> p, q;   // host copies
    char* block_dev = nullptr;  // one device allocation holding p, q, ctrl, stage_off, stage_len
    double* p_dev = nullptr;    // [n_p+1]
    double* q_dev = nullptr;    // [n_q+1]
    // Staged result of the last selection pass on this grid (scratch owned by the handle, written by wpcd_perm_count,
    // consumed by wpcd_perm_build): one slot per box-test candidate.  Mutable: the calls take a const handle (the lattice
    // does not change); include/wpcd.h says that count and build on one handle must not overlap in time.
    mutable int32_t* stage_col = nullptr;       // [stage_cap]  column index, or -1 for a rejected candidate
    mutable double4* stage_ext = nullptr;       // [stage_cap]  vertices of smallest / largest polar angle of Pi (survivors)
    int32_t* stage_off = nullptr;               // [n_p*n_q]    first slot of a geometric row
    int32_t* stage_len = nullptr;               // [n_p*n_q]    number of candidates of a geometric row
    int32_t* ctrl = nullptr;                    // [4] device: slot cursor, overflow flag, nnz_geo
    int32_t* ctrl_pinned = nullptr;             // [4] pinned host copy
    mutable cudaEvent_t count_event = nullptr;  // behind the read-back of the selection result
    mutable cudaEvent_t rowptr_event = nullptr; // behind the row-pointer expansion of the last count
    mutable cudaStream_t count_stream = nullptr;
    mutable int64_t stage_cap = 0;
    mutable bool stage_valid = false;
    mutable bool select_ready = false;          // kernel attributes set
    mutable int64_t stage_nnz_geo = 0;
};

// ---- tables of the coupled-channel fill --------------------------
// The moment row of a geometric element holds, (l, l') block after block, the distinct monomials
//   mu = (k, A):  P_k(x) cos^{A+1} sin^{l+l'-A+1} / (zeta1^{l'+1} zeta2^{l+1}),
// so all monomials of one row-channel momentum l are ONE contiguous range of the row (an "l-group").
// The contraction value[element][pair] = sum_m M[element][m] G[pair][m] runs on the FP64 tensor cores
// (mma.sync m8n8k4: 8 elements x 8 pairs x 4 monomials per step).  An ITEM is a set of at most 8 pairs (gamma, gamma')
// of one l-group with the same l' and exactly the same monomials, its tables in MMA fragment order:
//   idx   [4 kt]           positions of the item's monomials inside the l-group's range (padding repeats the last one)
//   g     [kt][n_pairs][4] B fragments: lane (lane/4 < n_pairs) holds G[pair lane/4][monomial 4 k + lane%4]  (0 where padded)
//   pairs [n_pairs]        (prefix of ncoupled over gamma, ncoupled(gamma), rank of gamma' in the row, gamma')
// The pairs are grouped by (l, l') -- the monomials of one (l, l') are ONE contiguous range of the moment row -- and all
// tables of a group form one blob [items | pairs | idx | g] (16-byte aligned pieces, offsets inside the blob) that the
// contraction kernel copies to shared memory verbatim.  A CTA takes (group, block of a few 32-element tiles of consecutive
// geometric elements), stages that range of the tiles' moments in shared memory and deals (item, tile) pieces to its
// warps.  The values of a pair for the elements of one geometric row are one run of CSR row (gamma, r) (DESIGN.md
// section 6: a row's entries are [gamma' rank][geometric entry]) and leave the warp through a small transposition
// buffer as coalesced stores.
struct wpcd_ct_item { int32_t n_pairs, kt, idx_off, g_off, pair_off, pad0, pad1, pad2; };     // offsets: elements of the group's arrays
struct wpcd_ct_group { int32_t mu_lo, n_mono, n_items, blob_off, blob_bytes, pairs_off, idx_off, g_off; };   // byte offsets; items at 0
constexpr size_t WPCD_CT_BLOB_BYTES = 16 * 1024;   // tables of one group (a single item may exceed it: then the group is that item)
constexpr int WPCD_CT_ELEMS = 32;        // elements of a geometric row per work unit

struct wpcd_channels {
    int model = 0;
    int n_ch = 0, n_pairs = 0;
    int64_t n_terms = 0;
    int64_t n_coef = 0;          // (pair, monomial) coefficients: terms of a pair with equal (l1 + l1', k) merged
    bool swave_single = false;   // one channel, one term k=l1=l1'=0, l=l'=0
    double g0 = 0.0;
    std::vector<int32_t> qn;     // [n_ch*6]
    std::vector<int32_t> channel_l;
    std::vector<int32_t> pair_gamma, pair_gammap, term_k, term_l1, term_l1p;
    std::vector<int64_t> term_ptr;
    std::vector<double> term_g;
    // moment tables
    int n_mu = 0;                 // length of a moment row (class blocks with padding)
    int k_max = 0, l_max = 0;
    int n_ll = 0, n_trip = 0;
    std::vector<int32_t> ll_pack;     // [n_ll]   l | l' << 8            distinct (l, l')
    std::vector<int32_t> trip_pack;   // [n_trip] k | ll << 8            distinct (k, l, l'), sorted by (ll, k)
    std::vector<int32_t> mu_pack;     // [n_mu]   trip | ab << 16
    std::vector<int32_t> mu_ib_pack;  // [n_mu]   (k IS + ll) | ab << 16: the triple resolved for moments2_kernel
    std::vector<int32_t> ab_pack;     // [n_ab]   (A+1) | (B+1) << 8       distinct exponent pairs of cos, sin
    int n_ab = 0;
    // contraction tables (host copies; the device copies sit in tables_dev)
    std::vector<wpcd_ct_group> ct_groups;
    std::vector<unsigned char> ct_blob;      // group after group
    int ct_nmono_max = 0, ct_blob_max = 0;   // largest monomial range / blob of a group
    int ct_ncoup_max = 0;                    // largest number of coupled channels of a row
    // device tables (one allocation, tables_dev; the typed pointers below point into it)
    unsigned char* tables_dev = nullptr;
    int32_t* ncoupled_dev = nullptr;          // [n_ch]   number of gamma' coupled to gamma
    int64_t* chan_off_dev = nullptr;          // [n_ch+1] prefix of ncoupled
    int32_t* coupled_gp_dev = nullptr;        // [n_pairs] gamma' of block t of channel gamma at chan_off[gamma] + t
    std::vector<int32_t> coupled_gp;
    int32_t* ll_pack_dev = nullptr;
    int32_t* trip_pack_dev = nullptr;
    int32_t* mu_pack_dev = nullptr;
    int32_t* mu_ib_pack_dev = nullptr;
    int32_t* ab_pack_dev = nullptr;
    wpcd_ct_group* ct_groups_dev = nullptr;
    unsigned char* ct_blob_dev = nullptr;
    std::vector<int32_t> ncoupled;
    int64_t total_coupled = 0;
    // blocked product: the gamma' coupled to gamma as runs of consecutive channels, (rank of the first, first gamma', length)
    std::vector<int32_t> run_ptr;             // [n_ch + 1]
    std::vector<int4> runs;
    int32_t* run_ptr_dev = nullptr;
    int4* runs_dev = nullptr;
    int first_gamma = -1, first_gp = 0;       // the first channel that has entries, and the first gamma' coupled to it
};

namespace wpcd_detail {

// Gauss-Legendre rule of one build, passed BY VALUE to the fill kernels (a __grid_constant__ parameter: every launch
// carries its own copy in its constant bank, so builds of different orders may overlap in time on one device).
struct QuadRule {
    double xi[WPCD_MAX_QUAD];
    double w[WPCD_MAX_QUAD];
    double invk[WPCD_MAX_K + 2];   // 1/k for the Legendre recurrence of the coupled fill
};

void set_error(const std::string& msg);
extern std::atomic<int64_t> g_launches;

// Test / diagnosis switches behind wpcd_debug_set (include/wpcd.h); 0 = the library's own choice.
struct DebugSwitches {
    std::atomic<int> spmv_lanes_per_row{0};      // 4 / 8 / 16 / 32: force the lanes-per-row variant of the CSR product
    std::atomic<int> spmv_no_pipeline{0};        // 1: never take the software-pipelined long-row variant
    std::atomic<int> no_pdl{0};                  // 1: launch the products without programmatic dependent launch
    std::atomic<int> chain_mode{0};              // 1: fused chain whenever the matrix fits on chip, 2: never
    std::atomic<int> blocked_no_mma{0};          // 1: the blocked product never takes the tensor-core pass (scalar passes of 8, 4, 2, 1 vectors)
    std::atomic<int> blocked_tile_doubles{0};    // > 0: size of the blocked product's x tile (small values exercise the chunked paths)
};
extern DebugSwitches g_debug;

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
    double* moments;     // [(chunk + 32) * n_mu], element-major (coupled channels only)
    int4* elem_rec;      // [nnz_geo] (first entry of the geometric row, its length, geometric column, row) (coupled channels only)
    unsigned int* counters;  // [n_chunks]: the work-queue ticket of each chunk's contraction launch
    int64_t n_chunks;
    int64_t chunk;       // geometric elements per moment chunk
    size_t bytes;
};
Workspace carve_workspace(const wpcd_channels* ch, int64_t nnz_geo, void* base);

// pattern.cu  (compiled with -fmad=false: the predicate is an IEEE contract)
cudaError_t ensure_stage(const wpcd_grid* g, int64_t want_cap);
cudaError_t launch_geo_select(const wpcd_grid* g, int32_t* geo_row_ptr_dev /* out: ptr */, cudaStream_t st);
cudaError_t launch_rowptr(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr_dev, int64_t* row_ptr_dev,
                          cudaStream_t st);
cudaError_t launch_geo_gather(const wpcd_grid* g, const int32_t* geo_row_ptr_dev, int32_t* geo_col, int32_t* geo_row,
                              double2* geo_phi, cudaStream_t st);

// fill.cu
cudaError_t launch_fill_swave(const wpcd_grid* g, const wpcd_channels* ch, int n_quad, int rule, const QuadRule& qr,
                              int64_t nnz_geo, const Workspace& ws, int32_t* col_idx, double* values, cudaStream_t st);
cudaError_t launch_fill_coupled(const wpcd_grid* g, const wpcd_channels* ch, int n_quad, bool split, const QuadRule& qr,
                                int64_t nnz_geo, const Workspace& ws, const int64_t* row_ptr, const int32_t* geo_row_ptr,
                                int32_t* col_idx, double* values, cudaStream_t st);

// spmv.cu
cudaError_t launch_spmv(int64_t rows, const int64_t* row_ptr, const int32_t* col_idx, const double* values,
                        const double* x, double* y, int n_vec, cudaStream_t st);
cudaError_t launch_spmv_interleaved(int64_t rows, const int64_t* row_ptr, const int32_t* col_idx, const double* values,
                                    const double* x, double* y, int n_vec, int n_inter, cudaStream_t st);
// api.cu: the dynamic shared-memory limit of a kernel belongs to the function (per device) and setting it REPLACES the value.
// This keeps the largest size ever asked for, under a lock: launches from several host threads with different sizes
// (two builds with different channel sets) cannot undercut each other between the attribute call and the launch.
cudaError_t raise_dyn_smem(const void* kernel, size_t bytes);
template <class K> inline cudaError_t raise_dyn_smem(K* kernel, size_t bytes) { return raise_dyn_smem(reinterpret_cast<const void*>(kernel), bytes); }
// spmv_blocked.cu
cudaError_t launch_spmv_blocked(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr, const int32_t* col_idx,
                                const double* values, const double* x, double* y, int n_vec, cudaStream_t st);
cudaError_t launch_spmv_blocked_noalloc(const wpcd_grid* g, const wpcd_channels* ch, const int32_t* geo_row_ptr, const int32_t* col_idx,
                                        const double* values, const double* x, double* y, int nv, cudaStream_t st);
cudaError_t launch_spmv_chain(int64_t rows, const int64_t* row_ptr, const int32_t* col_idx, const double* values,
                              const double* x, double* y, int n_iter, int64_t nnz, cudaStream_t st, int* fused);
cudaError_t run_fp64_peak(cudaStream_t st, double* flops_out);

// kernel_apply.cu
cudaError_t launch_block_apply(int n_ch, int n_p, int n_cols, const double* A, bool transpose, const double* X, double* Y, cudaStream_t st);
cudaError_t launch_diag_scale(int64_t n, const double* g, const double* x, double* y, cudaStream_t st);

}  // namespace wpcd_detail
