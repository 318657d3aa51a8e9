/* wpcd.h -- C-ABI of libwpcd: the permutation-operator matrix P0 of the
 * wave-packet continuum discretisation (arxiv 1404.5253) on one NVIDIA B200.
 *
 * What the library computes (citations are PAPER.md lines):
 *   P0 = matrix of P = P12 P23 + P13 P23 (eq. 2, l.62) in the lattice basis
 *   |X_ij^{gamma}> of eq. (6) (l.110): element (gamma,i,j ; gamma',i',j') is the
 *   integral (A15) (l.457) of the geometric coupling function G of (A3) (l.390)
 *   over the region where the cell D_ij of one Jacobi set overlaps the cell
 *   D_i'j' of the other (A7, l.416).  "Selection of the nonzero elements"
 *   (step 2, l.311) -> wpcd_perm_count; "calculation of the nonzero elements"
 *   (step 3, l.312) -> wpcd_perm_build; the product with a vector inside the
 *   iterative solution (step 5, l.314; sparse storage l.304) -> wpcd_perm_apply.
 *   Readings of every silent/garbled point: DESIGN.md section "Readings" (R1..R13).
 *
 * Conventions
 *   - plain C, no exceptions cross the boundary; every call returns a
 *     wpcd_status (0 = WPCD_OK, < 0 error) and wpcd_last_error() returns a
 *     thread-local message for the last failing call of the calling thread.
 *   - "host" pointers are ordinary CPU memory; "dev" pointers are CUDA device
 *     memory on the CURRENT device, owned by the caller (e.g. torch tensors).
 *     The library owns only the small tables inside its handles.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = default stream).
 *     All work is enqueued on it; only wpcd_perm_count synchronises (it must
 *     return nnz to the host).
 *   - index convention: cell (i,j), i = 0..n_p-1 the p-bin [p_i,p_{i+1}], j = 0..n_q-1
 *     the q-bin; geometric row r = i*n_q + j; full row = gamma*n_p*n_q + r; columns
 *     alike with primed indices; columns strictly ascending inside a row.
 *   - there is no CPU fallback: without a CUDA device every compute call
 *     returns WPCD_ERR_CUDA.
 *   - a GRID handle carries the staged result of its last selection pass (scratch written by wpcd_perm_count, read by
 *     wpcd_perm_build): the count and build calls on ONE grid handle must not overlap in time -- issue them from one
 *     thread, and let a build that is still running on its stream finish (or order the next count behind it on the
 *     same stream) before counting on that handle again.  Different grid handles, and any number of channel handles,
 *     may be used concurrently from different threads and streams (the quadrature rule travels with each launch).
 */
#ifndef WPCD_H
#define WPCD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wpcd_grid wpcd_grid;
typedef struct wpcd_channels wpcd_channels;
typedef int wpcd_status;

#define WPCD_OK 0
#define WPCD_ERR_INVALID_ARG (-1)   /* null pointer, non-positive size, bad enum */
#define WPCD_ERR_NOT_MONOTONE (-2)  /* nodes not strictly increasing or first node < 0 */
#define WPCD_ERR_ALLOC (-3)
#define WPCD_ERR_CUDA (-4)          /* CUDA runtime error or no device */
#define WPCD_ERR_OVERFLOW (-5)      /* column index would not fit int32 / nnz int64 */
#define WPCD_ERR_UNSUPPORTED (-6)   /* n_quad, l or k beyond WPCD_MAX_* */

#define WPCD_MAX_QUAD 64            /* Gauss-Legendre points per dimension (paper: 48, l.334) */
#define WPCD_RULE_KINK_SPLIT 0x100   /* OR into n_quad: the kink-split rule RS(n) of DESIGN.md R14 */
#define WPCD_RULE_ANALYTIC_U 0x200   /* OR into n_quad: rule RA(n) of DESIGN.md R15, exact x-integral; s-wave term only */
#define WPCD_MAX_L 7                /* largest pair orbital momentum l */
#define WPCD_MAX_K 23               /* largest Legendre order k in (A3) */

#define WPCD_SPINLESS_SWAVE 0       /* one channel l = lambda = 0, G = g0 (R4) */
#define WPCD_ND 1                   /* nucleon-deuteron channels of eq. (5), g from (A4) */

/* Message for the last error raised on this thread ("" if none). Static storage. */
const char* wpcd_last_error(void);

/* Momentum lattice: p_nodes[0..n_p] and q_nodes[0..n_q], HOST,
 * strictly increasing, first node >= 0, in fm^-1 (any unit: P0 is scale free).
 * Copies the nodes to the device.  *out is owned by the library. */
wpcd_status wpcd_grid_create(const double* p_nodes, int n_p, const double* q_nodes, int n_q, wpcd_grid** out);
void wpcd_grid_destroy(wpcd_grid* grid);

/* Channel set for fixed Gamma = {J, pi, T} (eq. 5, l.98-102) and its coefficient
 * table g^{l1 l1' k}_{gamma gamma'} of (A4) (l.395), computed on the host (step 1, l.310).
 *   model = WPCD_SPINLESS_SWAVE: two_J, parity, two_T, j_pair_max ignored; g = g0.
 *   model = WPCD_ND: parity = +1/-1, two_T = 1, pair momentum j <= j_pair_max; g0 ignored.
 * Channel order: ascending j, then s, then l, then two_I, then lambda
 * (channel = (l, s, j, t, lambda, two_I); t fixed by l+s+t odd, l.102).
 * Channel pairs whose every coefficient vanishes are not coupled and get no entries. */
wpcd_status wpcd_channels_create(int model, int two_J, int parity, int two_T, int j_pair_max, double g0,
                                 wpcd_channels** out);

/* Same, from a caller-supplied table (all HOST arrays): channel_l[n_channels] = l of each
 * channel; pair c = (pair_gamma[c], pair_gammap[c]) sorted ascending by (gamma, gamma'),
 * each pair once; its terms term_ptr[c] .. term_ptr[c+1]-1 are (k, l1, l1', g) multiplying
 * q^{l1+l1'} q'^{(l-l1)+(l'-l1')} P_k(x) in (A3) (reading R1). */
wpcd_status wpcd_channels_create_from_table(int n_channels, const int32_t* channel_l, int n_pairs,
                                            const int32_t* pair_gamma, const int32_t* pair_gammap,
                                            const int64_t* term_ptr, const int32_t* term_k,
                                            const int32_t* term_l1, const int32_t* term_l1p,
                                            const double* term_g, wpcd_channels** out);
void wpcd_channels_destroy(wpcd_channels* channels);

/* Introspection (host side, no device work). */
int wpcd_channels_count(const wpcd_channels* channels);            /* number of channels */
int wpcd_channels_pairs(const wpcd_channels* channels);            /* number of coupled pairs */
int64_t wpcd_channels_terms(const wpcd_channels* channels);        /* total (k,l1,l1') terms */
/* Sizes of the coupled fill (the roofline's algorithmic flop count): the number of distinct
 * monomials (l, l', l1+l1', k) of (A3) -- one moment per geometric element each -- and the number of
 * (pair, monomial) coefficients the g-contraction multiplies (terms of a pair with equal l1+l1' and k merged). */
int wpcd_channels_monomials(const wpcd_channels* channels);
int64_t wpcd_channels_coefficients(const wpcd_channels* channels);
/* quantum numbers [n_channels][6] = (l, s, j, t, lambda, two_I); zeros for a table-made set
 * except l.  HOST output. */
wpcd_status wpcd_channels_get_quantum_numbers(const wpcd_channels* channels, int32_t* out);
/* The table in the layout of wpcd_channels_create_from_table; HOST outputs sized by the
 * three counts above (term_ptr: n_pairs+1). */
wpcd_status wpcd_channels_get_table(const wpcd_channels* channels, int32_t* pair_gamma, int32_t* pair_gammap,
                                    int64_t* term_ptr, int32_t* term_k, int32_t* term_l1, int32_t* term_l1p,
                                    double* term_g);

/* rows = columns = n_channels * n_p * n_q;  geometric rows = n_p * n_q. */
int64_t wpcd_rows(const wpcd_grid* grid, const wpcd_channels* channels);
int64_t wpcd_geo_rows(const wpcd_grid* grid);

/* Step 2 (l.311): structural nonzeros.  A cell pair is a structural nonzero iff the
 * cells overlap with positive measure under (A2) -- predicate S of DESIGN.md R6, evaluated
 * in IEEE double without contraction; it does not depend on the channel pair or n_quad.
 *   geo_row_ptr_dev [n_p*n_q + 1] int32 dev, out: CSR row pointer of the geometric pattern
 *   row_ptr_dev     [rows + 1]    int64 dev, out: CSR row pointer of P0
 *   nnz_out, nnz_geo_out          host, out
 * The pass evaluates the predicate once and keeps its verdicts (one slot per candidate cell pair) in
 * scratch memory owned by the GRID handle, for the wpcd_perm_build that follows; the handle grows that
 * scratch on demand (a first call on a large lattice may run the pass twice).
 * Waits once, for the selection pass and the read-back of the two counts; the expansion to row_ptr_dev is queued on
 * the stream behind it and may still be running when the call returns (stream order covers every later use; a
 * wpcd_perm_build on another stream is ordered behind it by the library). */
wpcd_status wpcd_perm_count(const wpcd_grid* grid, const wpcd_channels* channels, int n_quad, void* cuda_stream,
                            int64_t* row_ptr_dev, int32_t* geo_row_ptr_dev, int64_t* nnz_out, int64_t* nnz_geo_out);

/* Scratch needed by wpcd_perm_build for a pattern with nnz_geo geometric entries
 * (geometric column / row / phi-range lists, and for coupled channels a block of monomial
 * moments of at most 64 MiB, 16 bytes per geometric entry and a few counters).  0 on invalid arguments. */
size_t wpcd_perm_workspace_bytes(const wpcd_channels* channels, int64_t nnz_geo);

/* Steps 2b+3 (l.312): column indices and values.
 *   row_ptr_dev, geo_row_ptr_dev   as written by wpcd_perm_count for the same arguments.  The verdicts staged
 *                                  in the grid handle by the last wpcd_perm_count on it are consumed here (the
 *                                  geometric pattern depends on the grid only, so any channel set may follow any
 *                                  count on the same grid); a handle that has not been counted yet runs the
 *                                  selection itself first (and then synchronises the stream once)
 *   workspace_dev                  >= wpcd_perm_workspace_bytes(channels, nnz_geo) bytes, dev, 256-byte aligned
 *   col_idx_dev [nnz] int32, values_dev [nnz] double: dev, out
 * Value = (d_i dbar_j d_i' dbar_j')^{-1/2} * double integral (A15) of F (A14) times the
 * channel-pair sum (A3), by the rule R(n_quad) of DESIGN.md R7: n_quad-point Gauss-Legendre
 * in phi over the angular extent of the overlap polygon, and at every phi-node n_quad-point
 * Gauss-Legendre in x over the closed-form support of F.  1 <= n_quad <= WPCD_MAX_QUAD.
 * n_quad | WPCD_RULE_KINK_SPLIT selects the kink-split rule RS(n_quad) of DESIGN.md R14 instead (the phi-range cut at
 * the rectangle-corner angles, the x-range at the crossings of the members of (A14)'s min / max; about ten times
 * the accuracy and ten times the cost of R(n_quad)); n_quad | WPCD_RULE_ANALYTIC_U the rule RA(n_quad) of R15 (the
 * same cuts, the x-integral of every piece in closed form; only for the s-wave channel set, WPCD_ERR_UNSUPPORTED
 * otherwise).  The pattern (wpcd_perm_count) does not depend on the rule.
 * Coupled channels: a channel pair may use any number of (k, l1+l1') monomials; WPCD_ERR_CUDA "invalid argument" if the
 * tables of one (l, l') exceed shared memory (more than ~2000 distinct monomials for one (l, l')) or if
 * (largest number of coupled channels of a row + 1) * nnz_geo reaches 2^31.
 * Asynchronous on the stream. */
wpcd_status wpcd_perm_build(const wpcd_grid* grid, const wpcd_channels* channels, int n_quad, void* cuda_stream,
                            const int64_t* row_ptr_dev, const int32_t* geo_row_ptr_dev,
                            void* workspace_dev, size_t workspace_bytes,
                            int32_t* col_idx_dev, double* values_dev);

/* y = P0 x for n_vec vectors (step 5, l.314; l.304).  x_dev[v*rows + c], y_dev[v*rows + r],
 * v = 0..n_vec-1 (vector-major), dev.  Any CSR arrays with int64 row_ptr / int32 col_idx (as produced above, or the
 * caller's own).  Asynchronous, capturable in a CUDA graph: the kernel variant (lanes per row) is chosen on the device
 * from the mean row length row_ptr[rows] / rows; nothing is read back and nothing is remembered between calls. */
wpcd_status wpcd_perm_apply(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                            const double* values_dev, const double* x_dev, double* y_dev, int n_vec,
                            void* cuda_stream);

/* y = P0 x for n_vec COMPLEX vectors (the transition operator is complex, P0 is real;
 * next step of SURVEY.md section 8(f)): x_dev / y_dev hold interleaved (re, im) doubles,
 * x_dev[2 * (v*rows + c)], 16-byte aligned, dev.  One 16-byte gather and two multiply-adds per entry.
 * Asynchronous. */
wpcd_status wpcd_perm_apply_complex(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                                    const double* values_dev, const double* x_dev, double* y_dev, int n_vec,
                                    void* cuda_stream);

/* y = P0 x for n_inter = 2 or 4 vectors stored INTERLEAVED, x_dev[c*n_inter + v] (two complex or four real
 * vectors for n_inter = 4): one gather of n_inter*8 bytes per entry instead of n_inter separate ones -- the
 * layout for many right-hand sides (P0 is reused for ~100 energies).  16-byte aligned, dev.
 * Asynchronous. */
wpcd_status wpcd_perm_apply_interleaved(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                                        const double* values_dev, const double* x_dev, double* y_dev, int n_inter,
                                        void* cuda_stream);

/* y = P0 x for a matrix built by wpcd_perm_build on (grid, channels), using its block structure: P0 = (channel coupling
 * mask) x (geometric pattern), i.e. row (gamma,i,j) holds, for every gamma' coupled to gamma, the same geometric columns
 * shifted by gamma' * n_p * n_q.  One CTA per geometric row (i,j) gathers the values of x at those columns for all
 * channels into shared memory once, and the n_channels rows of that (i,j) then stream only their VALUES: 8 bytes per
 * nonzero from HBM instead of the 12 of the general CSR product, and one gather per (channel, geometric entry) instead of
 * one per nonzero (the SpMV is HBM-bound).  Several vectors share one pass over the matrix: 3 - 8 go
 * through the FP64 tensor cores (values as A fragments, the planes of the x tile as B; n_channels <= 64, else scalar
 * passes of 8, 4), fewer through scalar passes of 2, 1; n_vec is cut into such passes.  A tensor-core pass works on an
 * interleaved copy of its x vectors held in stream-ordered scratch (cudaMallocAsync / cudaFreeAsync on cuda_stream,
 * 64 rows bytes, released behind the product; allowed during stream capture).
 * geo_row_ptr_dev as written by wpcd_perm_count, col_idx_dev / values_dev by wpcd_perm_build, for THESE handles (not
 * checked; row_ptr_dev is not read); x_dev, y_dev [n_vec][rows], dev, x_dev must not alias y_dev.  Each row is summed in a
 * fixed order (deterministic; agrees with wpcd_perm_apply to rounding).  Asynchronous.  At most 64 such products in
 * flight per device at a time (the work-queue counters are a ring). */
wpcd_status wpcd_perm_apply_blocked(const wpcd_grid* grid, const wpcd_channels* channels, const int64_t* row_ptr_dev,
                                    const int32_t* geo_row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                    const double* x_dev, double* y_dev, int n_vec, void* cuda_stream);

/* The same product for callers that must not allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): 1 <= n_vec <= 8 vectors in ONE tensor-core pass, whose scratch -- the interleaved copy of the x vectors,
 * 64 bytes per row -- lives in a fixed device array of the library (WPCD_NOALLOC_MAX_ROWS rows = 16 MiB, held by every GPU
 * that loads the library until the process exits) instead of a stream-ordered allocation.  The call makes no cudaMalloc,
 * cudaMallocAsync, cudaFree or other allocating call.  Arguments, layout and result as wpcd_perm_apply_blocked (same
 * kernel, same summation order: identical output for 3 <= n_vec <= 8).
 * WPCD_ERR_UNSUPPORTED if rows = n_channels * n_p * n_q > WPCD_NOALLOC_MAX_ROWS, n_channels > 64 or n_vec > 8 -- nothing is
 * launched then; use wpcd_perm_apply_blocked.
 * All calls on a device share the array: each call overwrites every word it later reads (nothing has to be cleared
 * between calls), but two calls that overlap on the GPU -- different streams without an ordering between them -- race on
 * it and give wrong results.  Calls on one stream are ordered and safe.  Asynchronous. */
#define WPCD_NOALLOC_MAX_ROWS 262144
wpcd_status wpcd_perm_apply_blocked_noalloc(const wpcd_grid* grid, const wpcd_channels* channels, const int64_t* row_ptr_dev,
                                            const int32_t* geo_row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                            const double* x_dev, double* y_dev, int n_vec, void* cuda_stream);

/* The dependent products of the simple iteration (paper step 5; Neumann terms):
 * y_k = P0 y_{k-1}, k = 1 .. n_iter, y_0 = x.  y_dev holds all iterates, y_dev[(k-1)*rows + r] = (P0^k x)[r], dev;
 * x_dev [rows], dev, must not overlap y_dev.  A matrix in the size window where it pays (about 1.6e4 <= nnz <=
 * 1.6e5 on a B200, measured: spmv_chain.cu) runs the whole chain in ONE cooperative launch -- row slices resident
 * in shared memory, a grid-wide barrier between products; any other matrix takes n_iter ordinary products on the
 * stream.  Either way a row is summed in a fixed lane order (deterministic), but the two orders differ, so results
 * agree to rounding, not bit for bit, across the two paths.  Reads the number of nonzeros back once per call (it
 * sizes the shared-memory slices): synchronises the stream, then queues the work.  At most 64 fused chains in flight per
 * device (the barrier counters are a ring). */
wpcd_status wpcd_perm_apply_chain(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                                  const double* values_dev, const double* x_dev, double* y_dev, int n_iter,
                                  void* cuda_stream);

/* Next step of SURVEY.md section 8(f): the kernel of eq. (12) in factored form.
 * wpcd_block_apply: for every channel gamma, Y_gamma = A_gamma X_gamma (transpose = 0) or A_gamma^T X_gamma
 * (transpose != 0), where X_gamma is the n_p x n_q block x_dev[(gamma*n_p + i)*n_q + j] of the vector and
 * a_dev[(gamma*n_p + k)*n_p + i] a real matrix acting on the pair index -- the rotation O of eq. (8)/(10)
 * or the pair interaction V1 in the scattering-wave-packet basis.  complex_vectors != 0:
 * x, y hold interleaved (re, im).  x_dev must not alias y_dev.  Dense products on the FP64 tensor cores.
 * Asynchronous. */
wpcd_status wpcd_block_apply(int n_channels, int n_p, int n_q, const double* a_dev, int transpose, const double* x_dev,
                             double* y_dev, int complex_vectors, void* cuda_stream);

/* y = O ( P0 ( O^T ( V1 ( G1 .* x ) ) ) ): one application of the kernel K = P V1 G1 of eq. (12) with
 * P = O P0 O^T (eq. 10).  o_dev, v_dev: [n_channels][n_p][n_p] real (V1 block-diagonal in the channel: the
 * uncoupled-pair case); g1_dev: [rows] complex diagonal (the channel resolvent, analytic in
 * the paper, an input here); x_dev, y_dev: [rows] complex; scratch_dev: 2*rows complex (4*rows doubles);
 * all complex arrays interleaved (re, im), 16-byte aligned, dev.  CSR arrays of P0 as produced above.
 * Asynchronous. */
wpcd_status wpcd_kernel_apply(int n_channels, int n_p, int n_q, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                              const double* values_dev, const double* o_dev, const double* v_dev, const double* g1_dev,
                              const double* x_dev, double* y_dev, double* scratch_dev, void* cuda_stream);

/* Third step of SURVEY.md section 8(f): "solution of the resulting matrix equation by iteration using the
 * Pade-approximant technique".  For u = b + K u (eq. 12 applied to the source column b) the
 * elastic amplitude is one element of u (eq. 13): a = sum_n a_n, a_n = (K^n b)[element].
 * wpcd_neumann_terms runs the iteration on the device (n_terms - 1 kernel applications) and returns the
 * complex terms a_0 .. a_{n_terms-1} in terms_host (HOST, interleaved).  scratch_dev: (8*rows + 2*n_terms)
 * doubles, 16-byte aligned, dev.  Synchronises the stream.
 * wpcd_pade_sum (host only) sums the series with Wynn's epsilon algorithm -- the diagonal Pade approximants
 * of sum_n a_n lambda^n at lambda = 1 -- which converges where the plain series does not. */
wpcd_status wpcd_neumann_terms(int n_channels, int n_p, int n_q, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                               const double* values_dev, const double* o_dev, const double* v_dev, const double* g1_dev,
                               const double* b_dev, int64_t element, int n_terms, double* terms_host, double* scratch_dev,
                               void* cuda_stream);
wpcd_status wpcd_pade_sum(const double* terms_host, int n_terms, double* sum_out);

/* Same product with HOST vectors: copies x_host -> x_dev (scratch, dev, n_vec*rows doubles),
 * applies, copies y_dev (scratch) -> y_host, then synchronises.  With more than 8 vectors the call pipelines chunks of 8
 * over two internal copy streams (upload of the next chunk, products of this one on the caller's stream and download of the
 * previous one overlap; the uploads start at once, without waiting for work queued earlier on the stream, so x_dev / y_dev
 * must not be in use by such work); one such call at a time per process.  Pinned host memory makes the copies asynchronous. */
wpcd_status wpcd_perm_apply_host(int64_t rows, const int64_t* row_ptr_dev, const int32_t* col_idx_dev,
                                 const double* values_dev, const double* x_host, double* y_host, int n_vec,
                                 double* x_dev, double* y_dev, void* cuda_stream);

/* wpcd_perm_apply_blocked with HOST vectors: copies x_host -> x_dev (scratch, dev, n_vec*rows doubles), applies, copies
 * y_dev (scratch) -> y_host, then synchronises.  Pinned host memory makes the copies asynchronous. */
wpcd_status wpcd_perm_apply_blocked_host(const wpcd_grid* grid, const wpcd_channels* channels, const int64_t* row_ptr_dev,
                                         const int32_t* geo_row_ptr_dev, const int32_t* col_idx_dev, const double* values_dev,
                                         const double* x_host, double* y_host, int n_vec, double* x_dev, double* y_dev,
                                         void* cuda_stream);

/* FP64 FMA microbenchmark (the roofline denominator of the fill kernel):
 * runs a dependent-chain-free DFMA loop on the whole chip and returns achieved FLOP/s
 * (2 per DFMA) in *flops_out (host).  Synchronises. */
wpcd_status wpcd_fp64_peak(void* cuda_stream, double* flops_out);

/* Stage tracing for the roofline report: when enabled, CUDA events are recorded on the
 * caller's stream around every kernel of wpcd_perm_count / wpcd_perm_build.
 * wpcd_trace_read synchronises those events, ADDS the elapsed milliseconds of each stage since
 * the last read into ms_out[WPCD_TRACE_STAGES] (host) and the launch counts into
 * launches_out[WPCD_TRACE_STAGES] (host, may be NULL), then clears the record. */
#define WPCD_TRACE_STAGES 6
#define WPCD_STAGE_GEO_COUNT 0   /* predicate, per-row counts, staged verdicts, scan (steps a1, a2) */
#define WPCD_STAGE_SCAN 1        /* geo_row_ptr -> row_ptr of the full matrix        (step a2) */
#define WPCD_STAGE_GEO_INDEX 2   /* compaction of the staged verdicts -> column list (step a3) */
#define WPCD_STAGE_FILL_SWAVE 3  /* single-channel quadrature fill        (step a4) */
#define WPCD_STAGE_MOMENTS 4     /* coupled channels: monomial moments    (step a4) */
#define WPCD_STAGE_CONTRACT 5    /* coupled channels: g-contraction+store (step a4) */
wpcd_status wpcd_trace_enable(int on);
wpcd_status wpcd_trace_read(double* ms_out, int64_t* launches_out);

/* Number of kernels the library has launched from this process (bench.py's gpu_launches). */
int64_t wpcd_launch_count(void);

/* Test and diagnosis switches (process-wide; the library reads no environment variable).  value 0 restores the
 * library's own choice.  Keys:
 *   "spmv_lanes_per_row"    4 / 8 / 16 / 32: force that lanes-per-row variant of wpcd_perm_apply
 *   "spmv_no_pipeline"      1: never take the software-pipelined long-row variant
 *   "no_pdl"                1: launch the products without programmatic dependent launch
 *   "chain_mode"            1: wpcd_perm_apply_chain fuses whenever the matrix fits on chip, 2: never fuses
 *   "blocked_tile_doubles"  > 0: size of the x tile of wpcd_perm_apply_blocked (small values exercise its chunked paths)
 *   "blocked_no_mma"        1: wpcd_perm_apply_blocked never takes the tensor-core pass (scalar passes of 8, 4, 2, 1 vectors)
 * WPCD_ERR_INVALID_ARG for an unknown key. */
wpcd_status wpcd_debug_set(const char* key, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* WPCD_H */
