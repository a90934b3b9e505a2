// aprod mode 1 and mode 2 (rows a3, a5-a8): Algorithms 1 and 2 of the paper
// on the tiled, attitude-binned layout of gsr_internal.h.
//
// One CTA runs one job = a run of tiles whose rows all start their attitude block inside one
// window of `win` knots per axis.  The CTA keeps in shared memory
//     xw[0 .. 3*win)          the attitude window of x (aprod1) or its accumulator (aprod2)
//     xw[3*win .. 3*win+I)    the whole instrumental block
// so the 18 irregular column accesses of a row never leave the SM; only the
// astrometric columns (5 per star, rows star-sorted inside a job) and the global column go
// to L1/L2.  The matrix itself is streamed once, coalesced, plane by plane.
#include "gsr_internal.h"

namespace gsr {

constexpr int TPB1 = 1024;               // aprod1: four tiles in flight per CTA (latency-bound)
constexpr int TPB2 = 512;                // aprod2: two tiles in flight (shared-memory-pipe-bound)

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

struct RowRegs {
    double v[NPAR];
    int32_t s, a;
    int32_t c[6];
};

// Streaming loads of one row, all 32 issued back to back (volatile asm keeps them together and
// ahead of their first use, so every thread has 224 bytes in flight).
__device__ __forceinline__ double ld_stream_f64(const double* p) {
    double v;
    asm volatile("ld.global.cs.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ int32_t ld_stream_s32(const int32_t* p) {
    int32_t v;
    asm volatile("ld.global.cs.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void load_row(const unsigned char* __restrict__ T, int lr, RowRegs& r) {
    r.s = ld_stream_s32((const int32_t*)(T + OFF_STAR) + lr);
    r.a = ld_stream_s32((const int32_t*)(T + OFF_ATT) + lr);
#pragma unroll
    for (int j = 0; j < 6; ++j) r.c[j] = ld_stream_s32((const int32_t*)(T + OFF_INSTR + j * R * 4) + lr);
#pragma unroll
    for (int k = 0; k < NPAR; ++k) r.v[k] = ld_stream_f64((const double*)(T + k * R * 8) + lr);
}

// ---- aprod1: y[i] = ca*y[i] + sum_k A[i,k] x[col(i,k)]  (Algorithm 1) --------------------
template <bool NORM, bool PERM>
__global__ void __launch_bounds__(TPB1) k_aprod1(const unsigned char* __restrict__ tiles,
                                                const Job* __restrict__ jobs,
                                                const double* __restrict__ x, double* __restrict__ y,
                                                const double* __restrict__ ca_p,
                                                double* __restrict__ partials,
                                                const uint32_t* __restrict__ perm, int64_t S,
                                                int64_t D, int I, int win,
                                                const int* __restrict__ stop) {
    if (stop && *stop) return;
    extern __shared__ double xw[];
    __shared__ double red[TPB1 / 32];
    const Job job = jobs[blockIdx.x];
    const double* xatt = x + 5 * S;
    const double* xins = x + 5 * S + 3 * D;
    // stage the attitude window (three axes) and the instrumental block
    for (int i = threadIdx.x; i < 3 * win; i += TPB1) {
        const int ax = i / win, j = i - ax * win;
        const int64_t knot = (int64_t)job.a0 + j;
        xw[i] = knot < D ? __ldg(xatt + ax * D + knot) : 0.0;
    }
    double* xi = xw + 3 * win;
    for (int i = threadIdx.x; i < I; i += TPB1) xi[i] = __ldg(xins + i);
    const double xg = __ldg(xins + I);
    const double ca = *ca_p;
    __syncthreads();

    const int sub = threadIdx.x / R, lr = threadIdx.x % R;
    double q = 0.0;
    for (int t = sub; t < job.ntiles; t += (TPB1 / R)) {
        const int64_t tile = (int64_t)job.tile0 + t;
        const unsigned char* T = tiles + tile * TILE_BYTES;
        RowRegs r;
        load_row(T, lr, r);
        const int64_t ri = tile * R + lr;
        int64_t ry = ri;
        bool live = true;
        if (PERM) {
            const uint32_t pe = __ldcs(perm + ri);
            live = pe != PERM_PAD;
            ry = pe;
        }
        const double yold = live ? y[ry] : 0.0;
        const double* xa = x + 5 * (int64_t)r.s;
        double sum = 0.0;
#pragma unroll
        for (int k = 0; k < 5; ++k) sum = fma(r.v[k], __ldg(xa + k), sum);
        const double* wa = xw + (r.a - job.a0);
#pragma unroll
        for (int ax = 0; ax < 3; ++ax)
#pragma unroll
            for (int j = 0; j < 4; ++j) sum = fma(r.v[5 + 4 * ax + j], wa[ax * win + j], sum);
#pragma unroll
        for (int j = 0; j < 6; ++j) sum = fma(r.v[17 + j], xi[r.c[j]], sum);
        sum = fma(r.v[23], xg, sum);
        const double ynew = fma(ca, yold, sum);
        if (live) y[ry] = ynew;
        if (NORM) q = fma(ynew, ynew, q);   // padding rows: y stays 0
    }
    if (NORM) {
        q = warp_sum(q);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = q;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tsum = 0.0;
#pragma unroll
            for (int w = 0; w < TPB1 / 32; ++w) tsum += red[w];
            partials[blockIdx.x] = tsum;
        }
    }
}

// ---- aprod2: x[col(i,k)] += A[i,k] * (y[i]*sy)  (Algorithm 2) ----------------------------
// attitude and instrumental blocks: shared-memory accumulators (privatised per job), flushed
// once per job with one global atomic per touched column; astrometric block: segmented warp
// reduction over the star-sorted rows, one global atomic per (warp, star, column); global
// column: register accumulation over the whole job, one atomic per job.
// SQUARE: accumulate A[i,k]^2 instead (column sums of squares for the preconditioner).
template <bool SQUARE, bool PERM>
__global__ void __launch_bounds__(TPB2) k_aprod2(const unsigned char* __restrict__ tiles,
                                                const Job* __restrict__ jobs,
                                                const double* __restrict__ y, double* __restrict__ x,
                                                const double* __restrict__ sy_p,
                                                const uint32_t* __restrict__ perm, int64_t S,
                                                int64_t D, int I, int win,
                                                const int* __restrict__ stop) {
    if (stop && *stop) return;
    extern __shared__ double xw[];
    __shared__ double red[TPB2 / 32];
    const Job job = jobs[blockIdx.x];
    const int nacc = 3 * win + I;
    for (int i = threadIdx.x; i < nacc; i += TPB2) xw[i] = 0.0;
    double* xi = xw + 3 * win;
    const double sy = SQUARE ? 1.0 : *sy_p;
    __syncthreads();

    const int sub = threadIdx.x / R, lr = threadIdx.x % R, lane = threadIdx.x & 31;
    double g = 0.0;
    for (int t = sub; t < job.ntiles; t += (TPB2 / R)) {
        const int64_t tile = (int64_t)job.tile0 + t;
        const unsigned char* T = tiles + tile * TILE_BYTES;
        RowRegs r;
        load_row(T, lr, r);
        const int64_t ri = tile * R + lr;
        double yv = 1.0;
        if (!SQUARE) {
            if (PERM) {
                const uint32_t pe = __ldcs(perm + ri);
                yv = pe != PERM_PAD ? y[pe] * sy : 0.0;
            } else {
                yv = __ldcs(y + ri) * sy;
            }
        }
#pragma unroll
        for (int k = 0; k < NPAR; ++k) r.v[k] = SQUARE ? r.v[k] * r.v[k] : r.v[k] * yv;

        // attitude: shared-memory accumulators
        double* wa = xw + (r.a - job.a0);
#pragma unroll
        for (int ax = 0; ax < 3; ++ax)
#pragma unroll
            for (int j = 0; j < 4; ++j) atomicAdd(wa + ax * win + j, r.v[5 + 4 * ax + j]);
        // instrumental
#pragma unroll
        for (int j = 0; j < 6; ++j) atomicAdd(xi + r.c[j], r.v[17 + j]);
        // global
        g += r.v[23];
        // astrometric: segmented reduction, rows are star-sorted
        const int32_t s_up = __shfl_up_sync(0xffffffffu, r.s, 1);
        const bool head = lane == 0 || s_up != r.s;
        const unsigned heads = __ballot_sync(0xffffffffu, head);
        if (heads == 1u) {   // the whole warp lies inside one star
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const double tsum = warp_sum(r.v[k]);
                if (lane == 0 && tsum != 0.0) atomicAdd(x + 5 * (int64_t)r.s + k, tsum);
            }
        } else {
            // segmented inclusive scan; the last lane of each segment holds its sum
            const unsigned below = heads & ((2u << lane) - 1u);        // heads at or below me
            const int seg_start = 31 - __clz(below);
            const bool tail = lane == 31 || ((heads >> (lane + 1)) & 1u);
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                double vsum = r.v[k];
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const double up = __shfl_up_sync(0xffffffffu, vsum, o);
                    if (lane - o >= seg_start) vsum += up;
                }
                if (tail && vsum != 0.0) atomicAdd(x + 5 * (int64_t)r.s + k, vsum);
            }
        }
    }
    // global column: one atomic per job
    g = warp_sum(g);
    if (lane == 0) red[threadIdx.x >> 5] = g;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tsum = 0.0;
#pragma unroll
        for (int w = 0; w < TPB2 / 32; ++w) tsum += red[w];
        if (tsum != 0.0) atomicAdd(x + 5 * S + 3 * D + I, tsum);
    }
    // flush the privatised accumulators
    double* xatt = x + 5 * S;
    for (int i = threadIdx.x; i < 3 * win; i += TPB2) {
        const double vacc = xw[i];
        if (vacc != 0.0) {
            const int ax = i / win, j = i - ax * win;
            atomicAdd(xatt + ax * D + job.a0 + j, vacc);   // knot < D whenever vacc != 0
        }
    }
    double* xins = x + 5 * S + 3 * D;
    for (int i = threadIdx.x; i < I; i += TPB2) {
        const double vacc = xi[i];
        if (vacc != 0.0) atomicAdd(xins + i, vacc);
    }
}

template <typename K>
static int set_smem(K kernel, int bytes) {
    GSR_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    return GSR_OK;
}

static int aprod1_smem(const gsr_matrix* A) {
    const int b = A->smem_bytes;
    return b;   // measured: 2 CTAs x 1024 threads (64 warps) beat 1 CTA with a larger L1
}

int configure_product_kernels(const gsr_matrix* A) {
    int b = aprod1_smem(A);
    GSR_TRY(set_smem(k_aprod1<true, false>, b));
    GSR_TRY(set_smem(k_aprod1<false, false>, b));
    GSR_TRY(set_smem(k_aprod1<false, true>, b));
    b = A->smem_bytes;
    GSR_TRY(set_smem(k_aprod2<false, false>, b));
    GSR_TRY(set_smem(k_aprod2<false, true>, b));
    GSR_TRY(set_smem(k_aprod2<true, false>, b));
    return GSR_OK;
}

int launch_aprod1(const gsr_matrix* A, const double* x, double* y, const double* ca,
                  double* partials, const int* stop, const uint32_t* perm, cudaStream_t s) {
    if (A->n_jobs == 0) return GSR_OK;
    const int64_t S = A->dims.n_stars, D = A->dims.n_dfa;
    const int I = (int)A->dims.n_instr;
    if (perm)
        k_aprod1<false, true><<<A->n_jobs, TPB1, aprod1_smem(A), s>>>(A->tiles, A->jobs, x, y, ca, nullptr,
                                                                    perm, S, D, I, A->win, stop);
    else if (partials)
        k_aprod1<true, false><<<A->n_jobs, TPB1, aprod1_smem(A), s>>>(A->tiles, A->jobs, x, y, ca, partials,
                                                                    nullptr, S, D, I, A->win, stop);
    else
        k_aprod1<false, false><<<A->n_jobs, TPB1, aprod1_smem(A), s>>>(A->tiles, A->jobs, x, y, ca, nullptr,
                                                                     nullptr, S, D, I, A->win, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_aprod2(const gsr_matrix* A, const double* y, double* x, const double* sy,
                  const int* stop, const uint32_t* perm, cudaStream_t s) {
    if (A->n_jobs == 0) return GSR_OK;
    const int64_t S = A->dims.n_stars, D = A->dims.n_dfa;
    const int I = (int)A->dims.n_instr;
    if (perm)
        k_aprod2<false, true><<<A->n_jobs, TPB2, A->smem_bytes, s>>>(A->tiles, A->jobs, y, x, sy, perm, S, D,
                                                                    I, A->win, stop);
    else
        k_aprod2<false, false><<<A->n_jobs, TPB2, A->smem_bytes, s>>>(A->tiles, A->jobs, y, x, sy, nullptr, S,
                                                                     D, I, A->win, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s) {
    if (A->n_jobs == 0) return GSR_OK;
    k_aprod2<true, false><<<A->n_jobs, TPB2, A->smem_bytes, s>>>(A->tiles, A->jobs, nullptr, q, nullptr,
                                                                nullptr, A->dims.n_stars, A->dims.n_dfa,
                                                                (int)A->dims.n_instr, A->win, nullptr);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

}  // namespace gsr

using namespace gsr;

extern "C" {

int gsr_aprod1(const gsr_matrix* A, const double* x_dev, double* y_dev, gsr_stream stream) {
    if (!A || !x_dev || (!y_dev && A->dims.n_rows > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    return launch_aprod1(A, x_dev, y_dev, A->coef_one, nullptr, nullptr, A->perm, (cudaStream_t)stream);
}

int gsr_aprod2(const gsr_matrix* A, const double* y_dev, double* x_dev, gsr_stream stream) {
    if (!A || !x_dev || (!y_dev && A->dims.n_rows > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    return launch_aprod2(A, y_dev, x_dev, A->coef_one, nullptr, A->perm, (cudaStream_t)stream);
}

}  // extern "C"
