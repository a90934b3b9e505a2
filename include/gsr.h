/*
 * gsr.h -- C ABI of libgsr_b200: the hot path of the Gaia AVU-GSR solver (arxiv 2212.11675)
 * on one NVIDIA B200 (sm_100a).  Plain C, no C++/torch types, no exceptions, nothing printed.
 *
 * The library solves  min_x || A x - b ||_2  (Eq. 1) with the paper's
 * column-preconditioned LSQR (PC-LSQR), A given in the paper's compressed
 * form: per observation row i
 *     star_idx[i]      the "number of the star"                     (first half of M_i)
 *     att_start[i]     index of the first attitude element, relative to an axis block
 *                      (second half of M_i; reading A3)
 *     instr_col[6i+j]  the six instrumental column positions          (I_c)
 *     values[24i+k]    A_d: 5 astrometric | 3x4 attitude | 6 instrumental | 1 global
 * Column of coefficient k of row i  (S stars, D = N_DFA knots per axis, I instrumental):
 *     k = 0..4    5*star_idx[i] + k
 *     k = 5..16   5S + ((k-5)/4)*D + att_start[i] + (k-5)%4
 *     k = 17..22  5S + 3D + instr_col[6i + k-17]
 *     k = 23      5S + 3D + I
 * n_cols = 5S + 3D + I + 1.
 *
 * Conventions
 *   - Every function returns 0 (GSR_OK) or a negative gsr_status; gsr_strerror() names it.
 *   - "hd" pointers may be HOST or DEVICE memory; the library detects which
 *     (cudaPointerGetAttributes).  Host buffers are staged through device memory owned by the
 *     handle; pinned host memory is copied asynchronously, pageable memory synchronously.
 *   - "dev" pointers must be device memory of the current device.
 *   - stream is a cudaStream_t passed as void* (NULL = legacy default stream).  Work is
 *     enqueued on it; only the functions documented as synchronising wait for it.
 *   - The handle owns all device memory it allocates (cudaMalloc) until gsr_matrix_destroy.
 *     Callers keep ownership of every array they pass and may free it once the call returned.
 *   - There is no CPU fallback: on a device that is not compute capability 10.x every entry
 *     point returns GSR_EUNSUPPORTED; without a CUDA device, GSR_ECUDA.
 */
#ifndef GSR_H
#define GSR_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gsr_matrix gsr_matrix; /* opaque, library-owned */
typedef struct gsr_comm gsr_comm;     /* opaque: one rank of a row-sharded solve (NCCL) */
typedef void* gsr_stream;             /* cudaStream_t */

typedef enum {
    GSR_OK = 0,
    GSR_EINVAL = -1,       /* null pointer, bad dims, index out of range, star_idx decreasing */
    GSR_ENOMEM = -2,       /* cudaMalloc failed */
    GSR_ECUDA = -3,        /* a CUDA runtime call failed (sticky error is cleared) */
    GSR_ESTATE = -4,       /* call not legal in the handle's state */
    GSR_EUNSUPPORTED = -5, /* device is not sm_100, size limit (see gsr_matrix_begin) or option */
    GSR_ERANGE = -6        /* GSR_OPT_DETERMINISTIC: a pass left the range of its fixed-point sums */
} gsr_status;

typedef struct {
    int64_t n_rows;  /* m  observations                                   */
    int64_t n_stars; /* S  -> 5*S astrometric columns  */
    int64_t n_dfa;   /* D  knots per axis -> 3*D attitude columns; D >= 4 */
    int64_t n_instr; /* I  instrumental columns, I >= 1                   */
    int32_t n_glob;  /* must be 1                           */
} gsr_dims;

typedef struct {
    int32_t istop;         /* 0..7, Paige-Saunders stop reason (C3)                */
    int32_t istop_natural; /* first of rules 1-6 that fired (0: none); differs from istop
                              only with GSR_OPT_FORCE_ITNLIM                                   */
    int64_t itn;           /* iterations done                                                  */
    int64_t itn_natural;   /* iteration at which istop_natural fired (0: none)                 */
    double rnorm;          /* ||b - A x||   estimate                                          */
    double arnorm;         /* ||A^T (b - A x)|| estimate                                      */
    double anorm;          /* Frobenius-norm estimate of the iterated matrix                   */
    double acond;          /* condition estimate                                               */
    double xnorm;          /* ||z||, norm of the iterate of the system actually iterated       */
    double bnorm;          /* ||b||                                                            */
} gsr_lsqr_result;

/* ---- matrix ingest (SURVEY/DESIGN row a0) -------------------- */

/* One-shot build.  Copies and re-lays the four arrays (hd: host or device) into the device
 * layout, validates them on the device, SYNCHRONISES the stream before returning.
 * Rows must be grouped by star: star_idx non-decreasing.  att_start in
 * [0, D-4]; instr_col in [0, I) (duplicates inside a row are legal and add).
 * Errors: GSR_EINVAL (nothing is leaked, *out = NULL), GSR_ENOMEM, GSR_ECUDA. */
int gsr_matrix_create(gsr_matrix** out, const gsr_dims* dims,
                      const int32_t* star_idx_hd,  /* [m]     */
                      const int32_t* att_start_hd, /* [m]     */
                      const int32_t* instr_col_hd, /* [m*6]   row-major */
                      const double* values_hd,     /* [m*24]  row-major, paper's A_d order */
                      gsr_stream stream);

/* Chunked build for systems whose caller-form arrays do not fit beside the device copy
 * (config 3: 67 GB): begin, append consecutive row ranges in order, finalize.
 * append: row0 must equal the number of rows appended so far; arrays cover nrows rows.
 * finalize synchronises, reports validation errors (GSR_EINVAL) and makes the handle usable.
 *
 * Size limits (checked by gsr_matrix_begin / gsr_matrix_create before any device work; tested in
 * tests/test_abi.py):
 *   GSR_EINVAL        n_rows < 0, n_stars < 1, n_dfa < 4, n_instr < 1, n_glob != 1;
 *                     n_cols = 5 S + 3 D + I + 1 >= 2^31 (int32 column indices);
 *                     n_rows >= 2^32 - 16 (uint32 row permutation; shard larger systems,
 *                     gsr_matrix_set_comm, or stream them, gsr_matrix_begin_streamed)
 *   GSR_EUNSUPPORTED  n_instr > 27 520: the product kernels keep the whole instrumental block of
 *                     x (8 I bytes) in shared memory beside 32 attitude windows (227 KB per SM);
 *                     more than 4096 attitude bins: n_dfa - 3 > 4096 * bw, where the bin width bw
 *                     (knots) is what fits in the per-warp window, bw = 241 for I <= 3 328
 *                     falling to 177 at I = 10 000 and 1 at I = 27 520, i.e. n_dfa <= 987 139 for
 *                     I <= 3 328 and n_dfa <= 724 995 at I = 10 000;
 *                     a device that is not sm_100.
 * All product and solve calls on one handle must be stream-ordered with respect to each other
 * (one stream, or events between streams): they share the handle's unit counter and workspace. */
int gsr_matrix_begin(gsr_matrix** out, const gsr_dims* dims, gsr_stream stream);

/* Out-of-core build ("1.8e9 rows": the system
 * "does not fit" one device).  As gsr_matrix_begin, but at most resident_bytes of the tiled
 * matrix stay in device memory; the rest is kept in PINNED HOST memory owned by the handle
 * (gsr_matrix_host_bytes) and crosses the bus once per pass over the matrix: every product,
 * gsr_precondition (which also writes the scaled tiles back) and every LSQR iteration stream
 * it through two device buffers of chunk_bytes each (raised to 1.7 MB if smaller), the H2D copy
 * of the next chunk overlapping the kernels of the current one.  append / finalize / products /
 * solve are used exactly as for a resident handle; results differ from a resident solve only
 * in the order of floating-point atomic adds.  The m-sized work vectors and the row
 * permutation (12 B/row) stay on the device.  If resident_bytes covers the whole matrix the
 * handle is an ordinary resident one.  Not combined with gsr_matrix_set_comm or
 * GSR_OPT_DETERMINISTIC (gsr_lsqr_solve: GSR_EUNSUPPORTED).
 * Errors: as gsr_matrix_begin; GSR_EINVAL for negative sizes; GSR_ENOMEM if the host memory
 * cannot be pinned. */
int gsr_matrix_begin_streamed(gsr_matrix** out, const gsr_dims* dims, int64_t resident_bytes,
                              int64_t chunk_bytes, gsr_stream stream);
int64_t gsr_matrix_host_bytes(const gsr_matrix* A);     /* pinned host memory owned by the handle */
int64_t gsr_matrix_streamed_bytes(const gsr_matrix* A); /* host-to-device bytes copied so far    */
int gsr_matrix_append_rows(gsr_matrix* A, int64_t row0, int64_t nrows,
                           const int32_t* star_idx_hd, const int32_t* att_start_hd,
                           const int32_t* instr_col_hd, const double* values_hd);
int gsr_matrix_finalize(gsr_matrix* A);

int gsr_matrix_destroy(gsr_matrix* A); /* NULL is legal */
int gsr_matrix_dims(const gsr_matrix* A, gsr_dims* out, int64_t* n_cols);
int64_t gsr_matrix_device_bytes(const gsr_matrix* A); /* device memory owned by the handle */

/* ---- the two products (rows a3, a5-a8; Algorithms 1 and 2) ----------- */

/* aprod mode 1:  y[i] = y[i] + sum_k A[i,k] x[col(i,k)]   ("b[i] = b[i] + sum").
 * x_dev [n_cols], y_dev [m], device pointers, caller-owned.  Asynchronous on stream. */
int gsr_aprod1(const gsr_matrix* A, const double* x_dev, double* y_dev, gsr_stream stream);

/* aprod mode 2:  x[col(i,k)] = x[col(i,k)] + A[i,k] y[i].
 * y_dev [m], x_dev [n_cols].  Asynchronous on stream.  Uses scratch inside the handle: calls
 * on the same handle must be stream-ordered.  In the default two-launch form
 * (GSR_OPT_APROD2_SPLIT) the first call allocates an m-sized work vector (8 bytes per row, y in
 * the internal row order; counted by gsr_matrix_device_bytes; GSR_ENOMEM if it does not fit). */
int gsr_aprod2(const gsr_matrix* A, const double* y_dev, double* x_dev, gsr_stream stream);

/* The same two products on vectors kept in the library's INTERNAL row order.  gsr_aprod1/2 take y
 * in the caller's row order and pay for it inside the kernel: the rows of a 32-row tile are
 * scattered over their ingest segment, so every tile gathers (scatters) its 32 entries of y one by
 * one -- measured at 3e8 rows 4.86 / 4.38 TB/s against 7.18 / 4.82 TB/s in the internal order
 * (profiles/r2_cfg5_sweep.md).  LSQR only ever touches m-sized vectors through A and A^T, so a
 * caller that iterates (the solver itself does this) converts ONCE and then runs every product at
 * the internal-order rate:
 *     gsr_matrix_internal_rows   length of an internal-order vector: the rows padded to whole
 *                                tiles per attitude bin, plus the constraint rows (-1 before
 *                                finalize)
 *     gsr_vector_to_internal     yint[i] = y[row of internal position i], 0 in padding positions
 *     gsr_vector_from_internal   the inverse; padding positions are dropped
 *     gsr_aprod1_internal        yint += A x      (Algorithm 1)
 *     gsr_aprod2_internal        x += A^T yint    (Algorithm 2)
 * Padding positions belong to all-zero rows: aprod1 leaves them as they are, aprod2 ignores them.
 * All pointers are device memory owned by the caller; asynchronous on `stream`; same stream-order
 * rule as the other products.  aprod2 runs as GSR_OPT_APROD2_SPLIT says. */
int64_t gsr_matrix_internal_rows(const gsr_matrix* A);
int gsr_vector_to_internal(const gsr_matrix* A, const double* y_dev, double* yint_dev, gsr_stream stream);
int gsr_vector_from_internal(const gsr_matrix* A, const double* yint_dev, double* y_dev, gsr_stream stream);
int gsr_aprod1_internal(const gsr_matrix* A, const double* x_dev, double* yint_dev, gsr_stream stream);
int gsr_aprod2_internal(const gsr_matrix* A, const double* yint_dev, double* x_dev, gsr_stream stream);

/* ---- preconditioner (row a1; Algorithm 3 line 2) ---------------------- */

/* p_j = 1/||A_j||_2 (1 for an empty column); every stored coefficient is multiplied by
 * p[col] in place; p is kept in the handle and, if p_out_hd != NULL, copied out ([n_cols],
 * host or device).  A second call returns GSR_ESTATE.  Asynchronous unless p_out_hd is host. */
int gsr_precondition(gsr_matrix* A, double* p_out_hd, gsr_stream stream);

/* ---- LSQR (rows a2, a4, a9-a12; Algorithm 3; C3) --------- */

/* Solves min ||A x - b||.  If A was preconditioned the iteration runs on A.diag(p) and the
 * returned x is p (.) z ("we re-multiply the solution ... by the preconditioning vector",
 * PAPER.md:67); the norms in *result refer to the system actually iterated.
 * b_hd [m] and x_hd [n_cols] may each be host or device.  itnlim >= 1.  atol, btol, conlim
 * as in Paige & Saunders; conlim = 0 disables rule 3.  SYNCHRONISES the stream: when it
 * returns, x and *result (host) are valid.  The whole iteration runs on the device from a
 * captured CUDA graph; the host only launches it. */
int gsr_lsqr_solve(gsr_matrix* A, const double* b_hd, double* x_hd, int64_t itnlim, double atol,
                   double btol, double conlim, gsr_lsqr_result* result, gsr_stream stream);

/* Standard errors of the unknowns of the LAST gsr_lsqr_solve on this handle ("Variances ...
 * computation", Algorithm 3 line 17; "the standard errors" are re-multiplied by p
 * like the solution).  The paper prints no formula; this is Paige & Saunders':
 * var_j = sum over the iterations of (w_j / rho)^2, accumulated inside the fused vector update,
 * se_j = p_j * rnorm * sqrt(var_j / max(m - n, 1)).  se_hd [n_cols], host or device.
 * GSR_ESTATE if no solve has finished on the handle.  Synchronises if se_hd is host memory. */
int gsr_lsqr_standard_errors(gsr_matrix* A, double* se_hd, gsr_stream stream);

/* ---- constraint equations (PAPER.md:65; "constraints computation", Algorithms 1-2, :280, :390) --
 * "To find a unique solution, an additional number of constraint equations have to be set."  The
 * paper does not give their structure: here they are n_con extra rows in general CSR form
 * appended BELOW the m observation rows (row m+r has val[e] at column col[e] for e in
 * [row_ptr[r], row_ptr[r+1]); columns in [0, n_cols)).  Arrays may be host or device and are
 * copied.  Call after create/finalize and before gsr_precondition / gsr_lsqr_solve; n_con = 0
 * removes them.  Afterwards every m-sized vector of the API (y of gsr_aprod1/2, b of
 * gsr_lsqr_solve) has m + n_con entries, observations first; gsr_precondition counts the
 * constraint coefficients in the column norms and scales them too.
 * On a row shard (gsr_matrix_set_comm) every constraint row is given to exactly ONE rank (rank 0
 * is the natural owner; the others pass none), in that rank's LOCAL column numbering: it may
 * touch the owner's own astrometric columns and any replicated column.  After
 * gsr_matrix_set_comm the call re-checks that n_rows_global still covers this rank's rows plus
 * n_con (GSR_EINVAL otherwise).  Constraint rows on a shard have run through the library only with
 * a one-rank communicator (no box with two GPUs was available); the world-2 case is covered by
 * tests/test_sharding_gloo.py on the CPU, which restates the recurrences and does not call it.
 * Errors: GSR_EINVAL (bad row_ptr, column out of range), GSR_ESTATE.  Synchronous. */
int gsr_matrix_set_constraints(gsr_matrix* A, int64_t n_con, const int64_t* row_ptr_hd,
                               const int32_t* col_hd, const double* val_hd);

/* ---- row-sharded solve over several GPUs (Fig. 2; Algorithm 3 lines 8-16) --
 * One process per GPU.  The observation rows are split into contiguous star-aligned blocks
 * (paper_2212_11675_b200/sharding.py); every rank builds an ORDINARY matrix from its block, with
 * its own stars renumbered from 0 and the same D and I.  The astrometric slice of every
 * n-vector is then distributed with the rows, the attitude + instrumental + global slice
 * (local columns [5*S_local, n_local)) is REPLICATED and summed over the ranks: the paper's
 * MPI reduce, here one ncclAllReduce(sum, fp64) of 3D + I + 2 values per iteration (the local
 * sum of u_hat^2 rides in the same buffer) and one of 2 scalars, both inside the CUDA graph.
 *   gsr_comm_unique_id  rank 0: fills id_out (>= 128 bytes); the caller broadcasts it
 *   gsr_comm_create     every rank, same id (collective: returns when all ranks have joined)
 *   gsr_matrix_set_comm after create/finalize, before gsr_precondition and gsr_lsqr_solve;
 *                       n_rows_global / n_cols_global are those of the whole system (standard
 *                       errors); n_rows_global counts the constraint rows of every rank too.
 *                       comm = NULL restores the single-GPU behaviour.
 * With a communicator gsr_precondition sums the column norms of the replicated slice over
 * the ranks, gsr_lsqr_solve returns the local x (replicated slice identical on every rank)
 * and the norms of the WHOLE system; only the fused iteration is supported.
 * NCCL is loaded with dlopen (GSR_EUNSUPPORTED if libnccl.so.2 cannot be found). */
int gsr_comm_unique_id(void* id_out, int64_t bytes);
int gsr_comm_create(gsr_comm** out, int rank, int world, const void* id_in, int64_t bytes);
int gsr_comm_destroy(gsr_comm* c);
int gsr_matrix_set_comm(gsr_matrix* A, gsr_comm* c, int64_t n_rows_global, int64_t n_cols_global);

/* Damped LSQR (Paige & Saunders' damp parameter; the paper's solver is undamped, damp = 0, the
 * default): the next solves on this handle minimise || [A; damp I] x - [b; 0] ||_2 (on the
 * column-scaled system if A was preconditioned); result->rnorm is then the norm of that
 * augmented residual.  damp >= 0, else GSR_EINVAL. */
int gsr_lsqr_set_damp(gsr_matrix* A, double damp);

/* Options (per handle). */
enum {
    GSR_OPT_FORCE_ITNLIM = 1, /* 1: rules 1-6 are evaluated and recorded in *_natural but only
                                 the iteration limit stops the loop (fixed-count mode, A9)    */
    GSR_OPT_DETERMINISTIC = 2, /* 1: gsr_lsqr_solve uses no floating-point atomics: every sum that
                                 leaves a warp (astrometric runs, attitude windows, global column,
                                 instrumental accumulators) is added to t = A^T u_hat as a 64-bit
                                 fixed-point integer, so two solves on the same handle give
                                 bit-identical x, norms and standard errors (the paper names its
                                 atomics as a weakness).  Needs a preconditioned
                                 matrix (the range of the sums rests on unit column norms), the
                                 fused iteration, no constraint rows, no communicator, no damping:
                                 otherwise gsr_lsqr_solve returns GSR_EUNSUPPORTED; GSR_ERANGE if a
                                 pass exceeded its range (norm of u_hat grew more than 128-fold
                                 beyond every earlier alpha and beta).  Each partial sum is rounded
                                 once to 2^-54 of that range.  gsr_aprod2 and gsr_precondition keep
                                 their fp64 atomics.  0 (default): fp64 atomics               */
    GSR_OPT_FUSED = 3,        /* 1 (default): one LSQR iteration reads the matrix ONCE -- u_hat =
                                 A v - (alpha/beta) u_hat and A^T u_hat are formed in the same
                                 pass, v = A^T u_hat / beta - beta v afterwards (same recurrences,
                                 DESIGN.md 5.4); 0: aprod1 then aprod2, two reads per iteration  */
    GSR_OPT_FIXED_POINT = 4,  /* 1 (default): on a column-scaled matrix the instrumental pass of
                                 the fused iteration accumulates in exact 64-bit fixed point
                                 with native 32-bit shared atomics (order-independent sums,
                                 normwise error <= n_j 2^-62 ||u|| per column); 0: fp64 atomics  */
    GSR_OPT_APROD2_SPLIT = 5, /* how aprod2 (gsr_aprod2 and the two-pass iteration) runs.  1 or -1
                                 (default): two launches -- astrometric + attitude + global blocks
                                 over 152 B of every row with 24 warps per SM, then the
                                 instrumental block over the instrumental planes alone (fp64
                                 adds for an arbitrary y, componentwise accuracy as before; the
                                 solver's own calls, which know ||y||, use the exact fixed-point
                                 pass of GSR_OPT_FIXED_POINT there); 0: one launch that does all
                                 four blocks (Algorithm 2 as one sweep).  Measured on B200, split
                                 against sweep: 14.0 / 14.8 ms at 3e8 rows x 10 000 instrumental
                                 columns, 4.2 / 5.5 ms at 1e8 x 6000, 4.9 / 9.6 ms at 1e8 x 60     */
    GSR_OPT_WHILE_GRAPH = 6   /* 1: the whole iteration loop of gsr_lsqr_solve is ONE CUDA graph
                                 launch -- a conditional WHILE node whose body is the iteration
                                 and whose condition a device kernel sets from the stop flag --
                                 so neither the stop decision nor a launch crosses to the host
                                 between iterations (config 1, launch-bound: measured 60.5 against
                                 59.0 us per iteration with per-iteration launches, i.e. no gain,
                                 DESIGN.md 5.6; immaterial at 1e8 rows and above).  Ignored with
                                 a communicator or on a streamed handle.  0 (default): one
                                 graph launch per iteration, the stop flag polled from pinned
                                 memory every 32 (fixed-count mode: 256) -- the default because
                                 Nsight Compute cannot see kernel nodes inside a graph that has
                                 conditional nodes, and the per-kernel evidence under profiles/
                                 is taken from the default path                                 */
};
int gsr_set_option(gsr_matrix* A, int key, int64_t value);

const char* gsr_strerror(int code);

/* ---- a norm for callers that cannot allocate (row a4; the norms of Algorithm 3) --
 * out_dev[0] = || v ||_2 of a device vector, by the same two-stage reduction the solver uses for
 * beta, alpha and ||w|| -- but WITHOUT a handle and without any allocation: no cudaMalloc, no
 * cudaFree, no allocating library routine, on the first call or any later one.
 *
 * Who needs this.  Everything else here draws its scratch from a handle, and a handle draws it
 * from cudaMalloc.  That is not available to (a) code that runs while the device is already full
 * -- a config-3 handle holds ~64 GB of tiles plus its work vectors, and a host framework's
 * caching allocator may own what is left, so a cudaMalloc either fails or forces that framework
 * to release its cache -- and (b) code on a latency path: cudaMalloc and cudaFree synchronise
 * the whole device and would stall a solve that is in flight on another stream.  Such a caller
 * (a convergence monitor, a residual check between solves, a plug-in that is handed buffers and
 * a stream and nothing else) passes the vector and one double of output; the partial sums live
 * in a fixed array inside the library image.
 *
 * Cost and limit.  The array is 33 024 bytes of device memory on EVERY GPU that loads the library,
 * held until the process exits.  It holds 4096 partial sums of 2^17 elements each:
 * len <= GSR_NORM2_STATIC_MAX_LEN = 2^29 (a 4 GiB vector; config 3 has 3e8 rows).  A longer
 * vector is refused with GSR_EUNSUPPORTED ("size") before anything is launched; split it and
 * combine the pieces as sqrt(a^2 + b^2).
 *
 * Sharing.  All calls on a device use the same array, and it keeps what the last call left.  The
 * one word that must start at zero (the ticket that elects the CTA doing the second stage) is
 * cleared on `stream` at the start of every call; the partial sums a call reads are those it has
 * just written.  Calls whose GPU work can OVERLAP -- two streams with no event between them, two
 * host threads -- race on the array and give wrong norms: keep all calls of a device on one
 * stream or order them with events.  (The solver's own norms do not use this array.)
 *
 * First call.  The first call on each device looks up the array's device address
 * (cudaGetSymbolAddress, with that device current) and checks that the device is sm_100; later
 * calls reuse it.  Make that first call during set-up, before any stream capture is begun.
 *
 * v_dev [len] device memory (may be NULL if len = 0: the norm is 0), out_dev [1] device memory,
 * both caller-owned.  Asynchronous on `stream`; equal input gives bit-equal output.
 * Errors: GSR_EINVAL (null pointer, len < 0), GSR_EUNSUPPORTED (len above the limit, device not
 * sm_100), GSR_ECUDA. */
#define GSR_NORM2_STATIC_MAX_LEN ((int64_t)1 << 29)
int gsr_norm2_static(const double* v_dev, int64_t len, double* out_dev, gsr_stream stream);

/* ---- test / measurement exports -------------------------------------------------------- */

/* The 24 (column, value) pairs of rows [row0, row0+nrows) in CALLER row order, read back from
 * the device layout (after preconditioning: the scaled values).  Host output arrays.
 * Synchronous.  Used by the "index construction bit-exact" parity test. */
int gsr_debug_expand_rows(const gsr_matrix* A, int64_t row0, int64_t nrows, int64_t* cols_host,
                          double* vals_host);

/* Average device time (ms, CUDA events on `stream`) of `reps` back-to-back launches of the
 * product kernels as the solver runs them (internal row order, fused coefficients):
 * which = 1: aprod1 (u <- A v - c u, + norm partials), which = 2: aprod2 (v += A^T u/beta),
 * which = 3: the fused pass of GSR_OPT_FUSED (u <- A v - c u and t += A^T u without the
 * instrumental block), which = 4: its instrumental pass.
 * The handle's LSQR work vectors are used as they are and results are discarded: call it AFTER
 * a gsr_lsqr_solve, so that they hold real data -- on the zero vectors of a fresh handle every
 * zero-valued atomic of aprod2 is skipped and the kernels look up to 15 % faster than they are.
 * Synchronous. */
int gsr_time_product(gsr_matrix* A, int which, int reps, float* ms_avg, gsr_stream stream);

/* One pass of the solver's fused iteration kernels (k_fused + its instrumental pass, with the
 * handle's GSR_OPT_FIXED_POINT setting) on CALLER-ordered vectors, so that exactly the kernels
 * of the timed loop can be compared with the oracle's two products at any size:
 *     y <- A x + ca * y      (Algorithm 1; y_dev[m] in/out, caller row order)
 *     t <- t + A^T y_new     (Algorithm 2; t_dev[n] in/out)
 * x_dev[n], y_dev[m], t_dev[n] are device arrays owned by the caller.  Uses (and overwrites) the
 * handle's LSQR work vectors: a previous solve's standard errors are lost.  Not available with
 * constraint rows or a communicator (GSR_EUNSUPPORTED).  Asynchronous on `stream`. */
int gsr_debug_fused_pass(gsr_matrix* A, const double* x_dev, double ca, double* y_dev,
                         double* t_dev, gsr_stream stream);

/* Device time (ms, CUDA events on the solve's stream) of the ITERATION LOOP of the last
 * gsr_lsqr_solve on this handle: from the first iteration's first kernel to the last iteration's
 * last one, without the initialisation (row a2) and the finalisation (row a12).  -1 before any
 * solve.  bench.py times "exactly K steps" with it. */
double gsr_lsqr_last_loop_ms(const gsr_matrix* A);

/* Number of iteration graphs captured on this handle so far.  Everything that is decided at
 * capture time (iteration form, instrumental-pass variant, deterministic mode, constraint rows,
 * communicator) is part of the graph's cache key; tests use this to check that changing such an
 * option between two solves really re-captures. */
int64_t gsr_debug_graph_builds(const gsr_matrix* A);

/* 1 if the iteration loop of the last gsr_lsqr_solve on this handle ran as ONE launch of the
 * conditional-WHILE graph (GSR_OPT_WHILE_GRAPH), 0 if it ran as one graph launch per iteration. */
int gsr_debug_while_graph(const gsr_matrix* A);

/* Number of kernel launches issued by this library since load (for bench.py's gpu_launches). */
int64_t gsr_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* GSR_H */
