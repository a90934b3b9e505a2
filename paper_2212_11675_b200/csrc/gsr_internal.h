// Internal declarations of libgsr_b200 (not part of the C ABI; see include/gsr.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <functional>
#include <vector>

#include "gsr.h"

namespace gsr {

// ---- device layout ------------------------------------
// Rows are stored in WARP TILES of R = 32 rows; a tile is one contiguous, 128-byte-aligned
// record that one warp streams.  Lane l of the warp is the HOME LANE of tile row l: the
// plane-major fields below (astro, instr, icol, glob, star) and the m-sized vectors are indexed
// by home lane, and rows are star-sorted along the home lanes.
//   astro [5][32] f64   plane-major: lane l reads consecutive addresses, 256 B per request
//   att   [8][2][12][2] f64  the 32x12 attitude block by ATTITUDE SLOT (h, q), h < 2, q < 16
//         (att_slot() maps a home lane to its slot): record (i, h) holds coefficient j of slots
//         (h, 2i) and (h, 2i+1) side by side, so that lane (h, j), j < 12, fetches 16 bytes per
//         request and the 24 lanes of a request cover 384 contiguous bytes = 3 whole lines.  A
//         lane ends up owning a COLUMN of the 32x12 block: coefficient j of the 16 slots of its
//         half.  aprod2 then adds slot after slot into the window with 12 lanes at 12 distinct
//         addresses (plain read-modify-write, no atomics); aprod1 forms the 12 products per
//         slot the same way and sums them over the lanes with fp64 tensor-core MMAs whose
//         constant operands select and add (reduce_slots() in gsr_aprod.cu).
//   instr [6][32] f64   plane-major
//   icol  [3][32] u32   instrumental columns, two u16 per word: columns 2k | 2k+1 << 16
//                       (I <= 65535 is implied by the shared-memory plan)
//   glob  [32] f64
//   star  [32] i32
//   aoff  [2][16] u8    att_start - a0 of the unit (offset inside the warp's window), by
//                       attitude slot; the window is at most 256 knots wide
//   a0    i32           first knot of the window (same for every tile of a unit)
//   cmask u32           bit q: the windows of slots (0, q) and (1, q) overlap (|da| < 4), so
//                       aprod2 must add them one after the other
//   iperm [32] u16      instrumental slot code of home lane l: sum_e slot(e) 6^e, where the
//                       caller's e-th instrumental entry sits in slot(e) of instr / icol.  The
//                       entries of a row are permuted among the six slots at ingest so that the
//                       16 rows of a half-warp spread over the shared-memory banks in every
//                       slot (k_permute_instr); only gsr_debug_expand_rows reads the code
//   padding up to                                                       6784 B = 212 B/row
//
// INTERNAL ROW ORDER.  LSQR only ever touches the m-sized vectors through A and A^T, so the
// solver is free to keep them in any row order.  Rows are ingested in segments of SEG rows;
// inside a segment they are stably partitioned by FINE ATTITUDE BIN (att_start / fw), which
// keeps the star grouping inside every bin.  A "unit" is a run of tiles of one (segment, bin):
// every attitude column its rows touch lies in a window of fw+3 knots per axis, a few KB that
// ONE WARP keeps privately in shared memory.  Warps are autonomous: a persistent grid of CTAs
// fetches units from a global counter, one unit per warp at a time; only the instrumental
// block (I doubles) is shared by the warps of a CTA.  perm[] maps an internal row to the
// caller's row (0xFFFFFFFF for the zero padding rows that round every bin up to whole tiles).
constexpr int R = 32;                        // rows per tile (one warp)
constexpr int NPAR = 24;
constexpr int OFF_ASTRO = 0;                 // byte offsets inside a tile record
constexpr int OFF_ATTV = 5 * R * 8;          // 1280
constexpr int OFF_INSTRV = OFF_ATTV + 12 * R * 8;   // 4352
constexpr int OFF_ICOL = OFF_INSTRV + 6 * R * 8;    // 5888 (instrumental values and columns are
                                                    //       adjacent: the instrumental pass of the
                                                    //       fused iteration reads only these 1920 B)
constexpr int OFF_GLOBV = OFF_ICOL + 6 * R * 2;     // 6272
constexpr int OFF_STAR = OFF_GLOBV + R * 8;         // 6528
constexpr int OFF_AOFF = OFF_STAR + R * 4;          // 6656
constexpr int OFF_A0 = OFF_AOFF + R;                // 6688: i32 first knot of the tile's window
constexpr int OFF_CMASK = OFF_A0 + 4;               // 6692
constexpr int OFF_IPERM = OFF_CMASK + 4;            // 6696
constexpr int TILE_BYTES = 6784;                    // 53 * 128
static_assert(OFF_IPERM + R * 2 <= TILE_BYTES && TILE_BYTES % 128 == 0, "tile record");
// attitude slot 16*h + q of home lane l.  The mapping is the one the MMA reduction of aprod1
// delivers its sums in (reduce_slots() in gsr_aprod.cu): lane l receives the sum of slot
//   h = bit 2 of l,  q = 8 * (bit 3 of l) + 2 * (l & 3) + (bit 4 of l XOR h).
// (A lane's MMA fragment holds the sums of slots (h, q) and (h, q ^ 1); which of the two lanes l,
// l ^ 16 takes which is free.  With the XOR the 16 lanes of a half-warp own slots 16h + q that
// are distinct modulo 16, so that the per-tile store of u_hat by slot, ysm[att_slot(lane)], is
// free of shared-memory bank conflicts.)
__host__ __device__ inline int att_slot(int l) {
    const int h = (l >> 2) & 1;
    return 16 * h + 8 * ((l >> 3) & 1) + 2 * (l & 3) + ((l >> 4) ^ h);
}
// byte offset of coefficient k (paper order) of home lane lr inside a tile record
__host__ __device__ inline int val_offset(int k, int lr) {
    if (k < 5) return OFF_ASTRO + (k * R + lr) * 8;
    if (k < 17) {
        const int sl = att_slot(lr), h = sl >> 4, q = sl & 15;
        return OFF_ATTV + ((((q >> 1) * 2 + h) * 12 + (k - 5)) * 2 + (q & 1)) * 8;
    }
    if (k < 23) return OFF_INSTRV + ((k - 17) * R + lr) * 8;
    return OFF_GLOBV + lr * 8;
}
// instrumental column j of home lane lr
__host__ __device__ inline int icol_offset(int j, int lr) {
    return OFF_ICOL + ((j >> 1) * R + lr) * 4 + (j & 1) * 2;
}

constexpr int64_t SEG = 1 << 22;             // rows per ingest segment
constexpr int NBIN_MAX = 4096;               // fine attitude bins
constexpr int NWARP = 16;                    // warps per product CTA
constexpr int TPB = NWARP * 32;
constexpr int SMEM_BUDGET = 224 * 1024;      // dynamic shared memory a product CTA may use
constexpr int WIN_BYTES_MAX = 6 * 1024;      // per-warp attitude window, 3 axes (the fused
                                             // iteration kernel keeps two of them per warp)
constexpr int UNIT_TILES_MAX = 128;          // tiles per unit (upper bound)
constexpr uint32_t PERM_PAD = 0xFFFFFFFFu;

struct Unit {
    int32_t tile0;    // first tile of the unit
    int32_t ntiles;   // tiles in the unit
    int32_t a0;       // first knot of the unit's attitude window
    int32_t pad_;
};

// A run of units and the storage their tiles are read from.  `base` is the address tile 0 WOULD
// have: a resident matrix passes its tile array, a streamed chunk (row f4(iii), below) passes
// buffer - t0 * TILE_BYTES, so that the kernels keep their global tile and row indices.
struct TileView {
    unsigned char* base;
    int u0, u1;          // units [u0, u1)
    int64_t t0, t1;      // tiles [t0, t1) = exactly the tiles of those units
};

// Out-of-core storage (row f4(iii); systems larger than the device).  Tiles
// [0, res_cap) stay in device memory, tiles [res_cap, n_tiles) in pinned host memory.  Every
// pass over the matrix handles the resident run of units with one launch and the rest in
// CHUNKS (runs of whole units, at most chunk_cap tiles) that a copy stream brings into one of
// two device buffers while the other is being consumed: H2D copy of chunk c+1 || kernels of
// chunk c.  All ordering is by events, the host never waits inside a pass; in fixed-count mode
// the solver enqueues several iterations per poll of the stop flag, so that the copy stream does
// not idle across the n-sized tail kernels and the host round trip between iterations either.
struct Chunk {
    int u0, u1;
    int64_t t0, t1;
};
struct StreamStore {
    bool on = false;
    int64_t res_cap = 0;                 // tiles kept on the device
    int64_t chunk_cap = 0;               // tiles per chunk buffer
    int64_t host_cap = 0;                // tiles of pinned host storage
    unsigned char* host = nullptr;       // tile res_cap + i at host + i * TILE_BYTES
    unsigned char* buf[2] = {nullptr, nullptr};
    unsigned char* seg = nullptr;        // ingest: the tiles of the segment being scattered
    int64_t seg_cap = 0;
    cudaStream_t copy = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, done[2] = {nullptr, nullptr}, fork = nullptr;
    int res_units = 0;                   // units [0, res_units) lie wholly below res_cap
    std::vector<Chunk>* chunks = nullptr;
    int64_t h2d_bytes = 0;               // bytes copied host -> device so far (bench.py)
    bool need_fork = true;               // the next pass must order its copies after the work queued on
                                         // the compute stream: set by ingest and by every pass that
                                         // wrote tiles back; read-only passes leave it false, so the
                                         // first copies of a pass overlap the tail of the previous one
};

// Device-resident LSQR scalars (row a9): every kernel of the iteration reads its coefficients
// from here, so the captured graph never needs host values.
struct LsqrState {
    // recurrences (C3)
    double alpha, beta, rhobar, phibar, anorm, ddnorm, xxnorm, z, cs2, sn2;
    double bnorm, rnorm, arnorm, acond, xnorm;
    double damp, res2;  // damping parameter (0: none) and the residual part held by its rows
    // coefficients consumed by the vector kernels
    double ca;         // aprod1: u_hat <- A v + ca * u_hat      (ca = -alpha/beta)
    double inv_beta;   // aprod2 input scale: v += A^T (u_hat * inv_beta)
    double vscale;     // prescale: v <- vscale * v              (-beta)
    double inv_alpha;  // update: v <- v * inv_alpha
    double t1, t2;     // update: x += t1 w ; w = v + t2 w
    double inv_rho;    // update: var += (w * inv_rho)^2
    // controls
    double atol, btol, ctol;
    long long itn, itnlim, itn_nat;
    int istop, istop_nat, stop, force, beta_pos, pad_;
    // GSR_OPT_DETERMINISTIC: exponent of the fixed-point scale of the NEXT fused pass (2^det_e
    // must exceed the norm of the u_hat that pass produces), its rigorous cap from ||A||_F,
    // the largest alpha / beta seen so far, and the flag raised when a pass exceeded its range
    int det, det_e, det_cap, det_fail;
    double det_max;
};

struct Workspace {
    double* u = nullptr;        // [m_int]  u_hat (unnormalised), INTERNAL row order
    double* v = nullptr;        // [n]
    double* w = nullptr;        // [n]
    double* x = nullptr;        // [n]  iterate z of the (scaled) system
    double* t = nullptr;        // [n]  A^T u_hat of the fused pass (zero between iterations)
    double* var = nullptr;      // [n]  sum over the iterations of (w_j / rho)^2 (row f1)
    bool solved = false;        // var / last_rnorm belong to a finished solve
    double last_rnorm = 0.0;
    double last_loop_ms = 0.0;  // device time of the iteration loop of the last solve
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    double* part_u = nullptr;   // [max(n_units, NB_N)] per-unit partial sums of u_hat^2
    double* part_v = nullptr;   // [NB_N]  (sharded: replicated slice only)
    double* part_w = nullptr;   // [NB_N]
    double* part_va = nullptr;  // [NB_N]  sharded: distributed (astrometric) slice of v^2 / w^2
    double* part_wa = nullptr;  // [NB_N]
    double* red = nullptr;      // [4] scalars that cross the ranks: sum v_a^2, sum w_a^2, sum b^2
    double* stage_m = nullptr;  // [m] staging for a host b
    double* stage_n = nullptr;  // [n] staging for a host x
    LsqrState* st = nullptr;
    int* stop_host = nullptr;   // pinned
    cudaGraphExec_t graph = nullptr;
    cudaStream_t graph_stream = nullptr;
    bool graph_valid = false;
    int graph_key = 0;          // options frozen into the captured graph (build_graph)
    int64_t graph_ncon = 0;
    void* graph_comm = nullptr;
    int graph_builds = 0;       // graphs captured so far (gsr_debug_graph_builds)
    cudaGraphExec_t wgraph = nullptr;   // the whole loop: a conditional WHILE node around the iteration
    bool wgraph_tried = false;  // (same cache key as `graph`; built with it)
    bool last_loop_while = false;   // the last solve ran as ONE launch of wgraph
};

}  // namespace gsr

struct gsr_matrix {
    gsr_dims dims;
    int64_t n_cols, off_att, off_instr, off_glob;
    // layout
    int nbins, bin_width, win;      // fine attitude bins; win = bin_width + 3 knots per axis
    int wstride;                    // doubles between the axes of a window in shared memory:
                                    // win rounded up to 4 mod 16, so that the 3 x 4 addresses
                                    // of a row fall into 12 distinct 8-byte banks
    int smem_bytes;                 // dynamic shared memory of the product kernels
    int smem_fused;                 // ... of the fused iteration kernel (two windows per warp)
    int ctas_per_sm;                // resident product CTAs per SM the shared-memory plan allows
    int grid1, grid2;               // persistent grids of aprod1 / aprod2
    int grid2_main;                 // ... of aprod2 without its instrumental block (split form)
    int grid_fused, grid_instr;     // ... of the fused iteration kernel / its instrumental pass
    int64_t tiles_cap, n_tiles;     // allocated / used tiles
    int64_t m_int;                  // n_tiles * R, length of internal-order vectors
    unsigned char* tiles;           // tiles_cap * TILE_BYTES
    uint32_t* perm;                 // [tiles_cap * R]
    gsr::Unit* units;               // device copy of the unit table
    int n_units;
    std::vector<gsr::Unit>* units_host;
    int* unit_counter;              // device: next unit to fetch (reset before every product)
    // ingest
    int64_t rows_appended;
    int64_t seg_fill, seg_cap;
    int32_t *st_star, *st_att, *st_instr;   // staging segment, caller form
    double* st_vals;
    int* seg_counts;                // [nbins * nblk] scratch of the partition
    int* seg_bin_rows;              // [nbins] + [nbins] padded starts (device), mirrored on host
    int* last_star;                 // device scalar: star of the last row of the previous segment
    int state;                      // 0 building, 1 ready
    cudaStream_t stream;
    double* p;                      // [n] preconditioner (nullptr until gsr_precondition)
    int* err;                       // device error word (validation)
    double* coef_one;               // device constants {1.0, 1.0}
    int64_t device_bytes;
    int opt_force_itnlim;
    int opt_two_pass;               // 1: aprod1 + aprod2 per iteration instead of the fused pass
    int opt_no_fixed;               // 1: fp64 atomics in the instrumental pass even when scaled
    int opt_deterministic;          // 1: no floating-point atomics anywhere in the iteration
    int opt_while;                  // 1: the whole loop as one conditional-WHILE graph launch
    int opt_aprod2_split;           // GSR_OPT_APROD2_SPLIT + 1: 0 = auto (default), 1 = one sweep, 2 = split
    double* yint;                   // [m_int] scaled y in internal order, written by the main
                                    // launch of a caller-order gsr_aprod2 (allocated on first use)
    double damp;                    // gsr_lsqr_set_damp (row f4); 0 = the paper's undamped LSQR
    int64_t n_con, con_nnz;         // row f3: constraint rows (CSR) appended below the observations
    int64_t* con_ptr;
    int32_t* con_col;
    double* con_val;
    gsr_comm* comm;                 // row e: this handle is one row shard (nullptr: whole system)
    int64_t m_global, n_global;     // rows / columns of the whole system (= local without comm)
    int sm_count;
    gsr::Workspace ws;
    gsr::StreamStore so;            // row f4(iii): out-of-core storage (so.on)
};

namespace gsr {

extern long long g_launches;
inline void count_launch(long long k = 1) { g_launches += k; }

#define GSR_CUDA_TRY(expr)                          \
    do {                                            \
        cudaError_t e__ = (expr);                   \
        if (e__ != cudaSuccess) {                   \
            cudaGetLastError();                     \
            return e__ == cudaErrorMemoryAllocation ? GSR_ENOMEM : GSR_ECUDA; \
        }                                           \
    } while (0)

#define GSR_TRY(expr)             \
    do {                          \
        int rc__ = (expr);        \
        if (rc__ != GSR_OK) return rc__; \
    } while (0)

int comm_allreduce_sum(gsr_comm* c, double* buf, size_t count, cudaStream_t s);
// constraint rows (gsr_constraints.cu); all are no-ops when the handle has none
constexpr int CON_GRID_MAX = 592;
int con_grid(const gsr_matrix* A);   // CTAs = partial sums of y^2 written by launch_con_aprod1
int launch_con_aprod1(const gsr_matrix* A, const double* x, double* ycon, const double* ca,
                      double* partial, const int* stop, cudaStream_t s);
int launch_con_aprod2(const gsr_matrix* A, const double* ycon, double* x, const double* sy,
                      const int* stop, cudaStream_t s);
int launch_con_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s);
int launch_con_scale(const gsr_matrix* A, const double* p, cudaStream_t s);
int launch_con_copy_sumsq(const gsr_matrix* A, const double* bcon, double* ucon, double* partial,
                          cudaStream_t s);
void free_constraints(gsr_matrix* A);
int dev_alloc(gsr_matrix* A, void** p, size_t bytes);
void dev_free(gsr_matrix* A, void* p, size_t bytes);
bool is_device_ptr(const void* p);
int ensure_workspace(gsr_matrix* A);
void free_workspace(gsr_matrix* A);

// product launchers (gsr_aprod.cu).  coef points to device doubles.  `perm` selects the row
// order of the m-sized vector: nullptr = internal order (the solver), A->perm = caller order.
//   aprod1: y[i] = (*ca) * y[i] + sum_k A[i,k] x[col];  if partials != nullptr, per-unit sums
//           of y_new^2 are written to partials[0..n_units).
int launch_aprod1(const gsr_matrix* A, const double* x, double* y, const double* ca,
                  double* partials, const int* stop, const uint32_t* perm, cudaStream_t s);
//   aprod2: x[col] += A[i,k] * (y[i] * (*sy))
//   ss (optional): device sum of y^2 over all rows -- the solver's own calls; lets the instrumental
//   block take the exact fixed-point pass on a column-scaled matrix (aprod2_two_launches)
int launch_aprod2(const gsr_matrix* A, const double* y, double* x, const double* sy,
                  const int* stop, const uint32_t* perm, cudaStream_t s, const double* ss = nullptr);
//   column sums of squares (preconditioner): q[col] += A[i,k]^2
int launch_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s);
// fused LSQR pass (one read of the matrix per iteration):
//   u[i] = (*ca) * u[i] + sum_k A[i,k] v[col]   (partials[unit] = sum of u_new^2)
//   t[col] += A[i,k] * u_new[i]                  for the astrometric, attitude and global blocks
// followed by the instrumental pass  t[off_instr + c] += A[i,17+j] * u[i]  over the
// instrumental planes only.  t must hold zeros (or the value to accumulate onto) on entry.
// det_e != nullptr (GSR_OPT_DETERMINISTIC): t is accumulated as 64-bit fixed-point integers
// with the scale 2^(61 - *det_e); launch_det_finish turns it back into doubles.
int launch_fused(const gsr_matrix* A, const double* v, double* u, const double* ca,
                 double* partials, double* t, const int* stop, const int* det_e, cudaStream_t s);
int launch_aprod2_instr(const gsr_matrix* A, const double* u, double* t, const double* ss,
                        const int* stop, int det, cudaStream_t s);   // ss: device sum of u^2 (or nullptr)
int launch_fused_streamed(const gsr_matrix* A, const double* v, double* u, const double* ca,
                          double* partials, double* t, const int* stop, cudaStream_t s);
int launch_det_finish(const gsr_matrix* A, double* t, const int* det_e, const double* ss,
                      const int* stop, cudaStream_t s);
int configure_product_kernels(gsr_matrix* A);
// aprod2 as two launches (main launch + instrumental pass)?  Default (auto): yes.  With 24 warps
// per CTA the main launch is 13 % faster than with 16, which the one-sweep kernel cannot have (its
// fp64 accumulators need 113 registers), and the compare-and-swap adds no longer share the LSU
// pipe with the attitude read-modify-writes.  Measured on B200 with real vectors, split against
// one sweep (ms): cfg3 14.0 / 14.8, cfg2 4.23 / 5.46, 1.28e8 rows x 600 columns 5.53 / 6.85,
// cfg4 (60 columns) 4.9 / 9.6.
// (the solver's aprod2 with a known norm: main launch + fixed-point instrumental pass)
inline bool aprod2_fixed_split(const gsr_matrix* A) { return A->p != nullptr && !A->opt_no_fixed; }
inline bool aprod2_is_split(const gsr_matrix* A) { return A->opt_aprod2_split != 1; }

// One pass over the matrix: f(view) for the resident run of units, then for every streamed
// chunk (double-buffered H2D copies on the copy stream, overlapped with f of the previous view).
// writeback: f modifies the tiles; streamed chunks are copied back to the host afterwards.
int for_each_view(gsr_matrix* A, cudaStream_t s, const std::function<int(const TileView&)>& f,
                  bool writeback = false);
void free_stream_store(gsr_matrix* A);

}  // namespace gsr
