// aprod mode 1 and mode 2 (rows a3, a5-a8): Algorithms 1 and 2 of the paper
// on the tiled structure-of-arrays layout of gsr_internal.h.
#include "gsr_internal.h"

namespace gsr {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- aprod1: y[i] = ca*y[i] + sum_k A[i,k] x[col(i,k)]  (Algorithm 1) --------------------
// One CTA per tile, one thread per row; every plane read is a coalesced 256 B warp request.
template <bool NORM>
__global__ void __launch_bounds__(R) k_aprod1(const unsigned char* __restrict__ tiles,
                                              const double* __restrict__ x, double* __restrict__ y,
                                              const double* __restrict__ ca_p,
                                              double* __restrict__ partials, int64_t m, int64_t S,
                                              int64_t D, int64_t I, const int* __restrict__ stop) {
    if (stop && *stop) return;
    const unsigned char* T = tiles + (int64_t)blockIdx.x * TILE_BYTES;
    const int lr = threadIdx.x;
    const int64_t row = (int64_t)blockIdx.x * R + lr;
    double v[NPAR];
#pragma unroll
    for (int k = 0; k < NPAR; ++k) v[k] = __ldcs((const double*)(T + k * R * 8) + lr);
    const int64_t s = __ldcs((const int32_t*)(T + OFF_STAR) + lr);
    const int64_t a = __ldcs((const int32_t*)(T + OFF_ATT) + lr);
    int32_t c[6];
#pragma unroll
    for (int j = 0; j < 6; ++j) c[j] = __ldcs((const int32_t*)(T + OFF_INSTR + j * R * 4) + lr);
    const double yold = (row < m) ? y[row] : 0.0;
    const double* xa = x + 5 * s;
    const double* xt = x + 5 * S + a;
    const double* xi = x + 5 * S + 3 * D;
    double sum = 0.0;
#pragma unroll
    for (int k = 0; k < 5; ++k) sum = fma(v[k], __ldg(xa + k), sum);
#pragma unroll
    for (int ax = 0; ax < 3; ++ax)
#pragma unroll
        for (int j = 0; j < 4; ++j) sum = fma(v[5 + 4 * ax + j], __ldg(xt + ax * D + j), sum);
#pragma unroll
    for (int j = 0; j < 6; ++j) sum = fma(v[17 + j], __ldg(xi + c[j]), sum);
    sum = fma(v[23], __ldg(xi + I), sum);
    const double ynew = fma(*ca_p, yold, sum);
    if (row < m) y[row] = ynew;
    if (NORM) {
        __shared__ double red[R / 32];
        double q = (row < m) ? ynew * ynew : 0.0;
        q = warp_sum(q);
        if ((lr & 31) == 0) red[lr >> 5] = q;
        __syncthreads();
        if (lr == 0) {
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < R / 32; ++w) t += red[w];
            partials[blockIdx.x] = t;
        }
    }
}

// ---- aprod2: x[col(i,k)] += A[i,k] * (y[i]*sy)  (Algorithm 2) ----------------------------
// v0: astrometric block by warp reduction when the warp lies inside one star (rows are
// star-sorted), otherwise per-lane atomics; attitude / instrumental by L2 atomics (red.f64);
// global column by warp reduction + one atomic per warp.
// SQUARE: accumulate A[i,k]^2 instead (column sums of squares for the preconditioner).
template <bool SQUARE>
__global__ void __launch_bounds__(R) k_aprod2(const unsigned char* __restrict__ tiles,
                                              const double* __restrict__ y, double* __restrict__ x,
                                              const double* __restrict__ sy_p, int64_t m, int64_t S,
                                              int64_t D, int64_t I, const int* __restrict__ stop) {
    if (stop && *stop) return;
    const unsigned char* T = tiles + (int64_t)blockIdx.x * TILE_BYTES;
    const int lr = threadIdx.x;
    const int lane = lr & 31;
    const int64_t row = (int64_t)blockIdx.x * R + lr;
    double v[NPAR];
#pragma unroll
    for (int k = 0; k < NPAR; ++k) v[k] = __ldcs((const double*)(T + k * R * 8) + lr);
    const int32_t s = __ldcs((const int32_t*)(T + OFF_STAR) + lr);
    const int64_t a = __ldcs((const int32_t*)(T + OFF_ATT) + lr);
    int32_t c[6];
#pragma unroll
    for (int j = 0; j < 6; ++j) c[j] = __ldcs((const int32_t*)(T + OFF_INSTR + j * R * 4) + lr);
    double yv;
    if (SQUARE) yv = 1.0;
    else yv = (row < m) ? __ldcs(y + row) * (*sy_p) : 0.0;
#pragma unroll
    for (int k = 0; k < NPAR; ++k) v[k] = SQUARE ? v[k] * v[k] : v[k] * yv;

    // astrometric
    const int32_t s0 = __shfl_sync(0xffffffffu, s, 0);
    const bool uniform = __all_sync(0xffffffffu, s == s0);
    double* xa = x + 5 * (int64_t)s;
    if (uniform) {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            double t = warp_sum(v[k]);
            if (lane == 0) atomicAdd(xa + k, t);
        }
    } else {
#pragma unroll
        for (int k = 0; k < 5; ++k) atomicAdd(xa + k, v[k]);
    }
    // attitude
    double* xt = x + 5 * S + a;
#pragma unroll
    for (int ax = 0; ax < 3; ++ax)
#pragma unroll
        for (int j = 0; j < 4; ++j) atomicAdd(xt + ax * D + j, v[5 + 4 * ax + j]);
    // instrumental
    double* xi = x + 5 * S + 3 * D;
#pragma unroll
    for (int j = 0; j < 6; ++j) atomicAdd(xi + c[j], v[17 + j]);
    // global
    double g = warp_sum(v[23]);
    if (lane == 0) atomicAdd(xi + I, g);
}

int launch_aprod1(const gsr_matrix* A, const double* x, double* y, const double* ca,
                  double* partials, const int* stop, cudaStream_t s) {
    if (A->n_tiles == 0) return GSR_OK;
    if (partials)
        k_aprod1<true><<<(unsigned)A->n_tiles, R, 0, s>>>(A->tiles, x, y, ca, partials, A->dims.n_rows,
                                                          A->dims.n_stars, A->dims.n_dfa,
                                                          A->dims.n_instr, stop);
    else
        k_aprod1<false><<<(unsigned)A->n_tiles, R, 0, s>>>(A->tiles, x, y, ca, nullptr, A->dims.n_rows,
                                                           A->dims.n_stars, A->dims.n_dfa,
                                                           A->dims.n_instr, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_aprod2(const gsr_matrix* A, const double* y, double* x, const double* sy,
                  const int* stop, cudaStream_t s) {
    if (A->n_tiles == 0) return GSR_OK;
    k_aprod2<false><<<(unsigned)A->n_tiles, R, 0, s>>>(A->tiles, y, x, sy, A->dims.n_rows,
                                                       A->dims.n_stars, A->dims.n_dfa,
                                                       A->dims.n_instr, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s) {
    if (A->n_tiles == 0) return GSR_OK;
    k_aprod2<true><<<(unsigned)A->n_tiles, R, 0, s>>>(A->tiles, nullptr, q, nullptr, A->dims.n_rows,
                                                      A->dims.n_stars, A->dims.n_dfa,
                                                      A->dims.n_instr, nullptr);
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
    return launch_aprod1(A, x_dev, y_dev, A->coef_one, nullptr, nullptr, (cudaStream_t)stream);
}

int gsr_aprod2(const gsr_matrix* A, const double* y_dev, double* x_dev, gsr_stream stream) {
    if (!A || !x_dev || (!y_dev && A->dims.n_rows > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    return launch_aprod2(A, y_dev, x_dev, A->coef_one, nullptr, (cudaStream_t)stream);
}

}  // extern "C"
