// Internal declarations of libgsr_b200 (not part of the C ABI; see include/gsr.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "gsr.h"

namespace gsr {

// ---- device layout ------------------------------------
// Rows are stored in tiles of R rows; a tile is one contiguous record, plane-major:
//   val[24][R] f64 | att[R] i32 | star[R] i32 | instr[6][R] i32     = 224*R bytes
// so that lane r of a warp reads consecutive addresses in every plane (coalesced 256 B per
// warp request) and a whole tile is one contiguous stream for the memory system.
//
// INTERNAL ROW ORDER.  LSQR only ever touches the m-sized vectors through A and A^T, so the
// solver is free to keep them in any row order.  Rows are ingested in segments of SEG rows;
// inside a segment they are stably partitioned by ATTITUDE BIN (att_start / bin_width), which
// keeps the star grouping inside every bin.  A "job" is a run of tiles of one (segment, bin):
// every attitude column its rows touch lies in a window of bin_width+3 knots per axis, small
// enough to live in shared memory together with the whole instrumental block.  perm[] maps
// an internal row to the caller's row (0xFFFFFFFF for the zero padding rows that round every
// bin up to whole tiles).
constexpr int R = 256;                       // rows per tile
constexpr int NPAR = 24;
constexpr int OFF_ATT = NPAR * R * 8;        // byte offsets inside a tile record
constexpr int OFF_STAR = OFF_ATT + R * 4;
constexpr int OFF_INSTR = OFF_STAR + R * 4;
constexpr int TILE_BYTES = OFF_INSTR + 6 * R * 4;  // 57344
static_assert(TILE_BYTES == 224 * R, "tile record is 224 bytes per row");

constexpr int64_t SEG = 1 << 22;             // rows per ingest segment
constexpr int NBIN_MAX = 256;                // attitude bins
constexpr int SMEM_BUDGET = 220 * 1024;      // bytes of shared memory a product CTA may use
constexpr int ATT_WIN_BYTES = 64 * 1024;     // target size of the attitude window (3 axes)
constexpr int JOB_TILES_MAX = 128;           // tiles per job (upper bound)
constexpr uint32_t PERM_PAD = 0xFFFFFFFFu;

struct Job {
    int32_t tile0;    // first tile of the job
    int32_t ntiles;   // tiles in the job
    int32_t a0;       // first knot of the attitude window
    int32_t pad_;
};

// Device-resident LSQR scalars (row a9): every kernel of the iteration reads its coefficients
// from here, so the captured graph never needs host values.
struct LsqrState {
    // recurrences (C3)
    double alpha, beta, rhobar, phibar, anorm, ddnorm, xxnorm, z, cs2, sn2;
    double bnorm, rnorm, arnorm, acond, xnorm;
    // coefficients consumed by the vector kernels
    double ca;         // aprod1: u_hat <- A v + ca * u_hat      (ca = -alpha/beta)
    double inv_beta;   // aprod2 input scale: v += A^T (u_hat * inv_beta)
    double vscale;     // prescale: v <- vscale * v              (-beta)
    double inv_alpha;  // update: v <- v * inv_alpha
    double t1, t2;     // update: x += t1 w ; w = v + t2 w
    // controls
    double atol, btol, ctol;
    long long itn, itnlim, itn_nat;
    int istop, istop_nat, stop, force, beta_pos, pad_;
};

struct Workspace {
    double* u = nullptr;        // [m_int]  u_hat (unnormalised), INTERNAL row order
    double* v = nullptr;        // [n]
    double* w = nullptr;        // [n]
    double* x = nullptr;        // [n]  iterate z of the (scaled) system
    double* part_u = nullptr;   // [max(n_jobs, NB_N)] per-CTA partial sums of u_hat^2
    double* part_v = nullptr;   // [NB_N]
    double* part_w = nullptr;   // [NB_N]
    double* stage_m = nullptr;  // [m] staging for a host b
    double* stage_n = nullptr;  // [n] staging for a host x
    LsqrState* st = nullptr;
    int* stop_host = nullptr;   // pinned
    cudaGraphExec_t graph = nullptr;
    cudaStream_t graph_stream = nullptr;
    bool graph_valid = false;
};

}  // namespace gsr

struct gsr_matrix {
    gsr_dims dims;
    int64_t n_cols, off_att, off_instr, off_glob;
    // layout
    int nbins, bin_width, win;      // attitude bins; win = bin_width + 3 knots per axis
    int smem_bytes;                 // dynamic shared memory of the product kernels
    int64_t tiles_cap, n_tiles;     // allocated / used tiles
    int64_t m_int;                  // n_tiles * R, length of internal-order vectors
    unsigned char* tiles;           // tiles_cap * TILE_BYTES
    uint32_t* perm;                 // [tiles_cap * R]
    gsr::Job* jobs;                 // device copy of the job table
    int n_jobs;
    std::vector<gsr::Job>* jobs_host;
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
    int sm_count;
    gsr::Workspace ws;
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

int dev_alloc(gsr_matrix* A, void** p, size_t bytes);
void dev_free(gsr_matrix* A, void* p, size_t bytes);
bool is_device_ptr(const void* p);
int ensure_workspace(gsr_matrix* A);
void free_workspace(gsr_matrix* A);

// product launchers (gsr_aprod.cu).  coef points to device doubles.  `perm` selects the row
// order of the m-sized vector: nullptr = internal order (the solver), A->perm = caller order.
//   aprod1: y[i] = (*ca) * y[i] + sum_k A[i,k] x[col];  if partials != nullptr, per-job sums
//           of y_new^2 are written to partials[0..n_jobs).
int launch_aprod1(const gsr_matrix* A, const double* x, double* y, const double* ca,
                  double* partials, const int* stop, const uint32_t* perm, cudaStream_t s);
//   aprod2: x[col] += A[i,k] * (y[i] * (*sy))
int launch_aprod2(const gsr_matrix* A, const double* y, double* x, const double* sy,
                  const int* stop, const uint32_t* perm, cudaStream_t s);
//   column sums of squares (preconditioner): q[col] += A[i,k]^2
int launch_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s);
int configure_product_kernels(const gsr_matrix* A);

}  // namespace gsr
