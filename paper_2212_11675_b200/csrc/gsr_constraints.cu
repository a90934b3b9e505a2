// Row f3: constraint equations.  "To find a unique solution, an additional number of constraint
// equations have to be set"; both aprod modes of the paper end with a
// "constraints computation" (Algorithms 1 and 2) that it leaves on
// the CPU because it is 100-1000x cheaper than the products.  The paper does not
// give their structure, so they are n_con extra rows in general CSR form appended below the m
// observation rows; m-sized vectors then carry n_con more entries at the end.
// One CTA per constraint row (at most CON_GRID_MAX CTAs, grid-stride over the rows), block
// reductions in a fixed order, one partial sum of y^2 per CTA: deterministic for a given system.
#include <vector>

#include "gsr_internal.h"

namespace gsr {

__device__ __forceinline__ double wsum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

constexpr int CON_TPB = 256;

// deterministic block sum (fixed order): valid in thread 0
__device__ __forceinline__ double con_block_sum(double v, double* red) {
    v = wsum(v);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < CON_TPB / 32; ++w) t += red[w];
    __syncthreads();
    return t;
}

// One CTA per constraint row (grid-stride over the rows), the row's entries strided over the
// threads: y[r] = ca*y[r] + sum_e val[e] x[col[e]]; partial[blockIdx.x] = sum over the CTA's
// rows of y_new[r]^2 (if partial != nullptr).  Fixed summation order for a fixed grid.
__global__ void __launch_bounds__(CON_TPB) k_con_aprod1(int64_t n_con, const int64_t* __restrict__ ptr,
                                                        const int32_t* __restrict__ col,
                                                        const double* __restrict__ val,
                                                        const double* __restrict__ x, double* __restrict__ y,
                                                        const double* __restrict__ ca_p,
                                                        double* __restrict__ partial,
                                                        const int* __restrict__ stop) {
    if (stop && *stop) return;
    __shared__ double red[CON_TPB / 32];
    const double ca = *ca_p;
    double q = 0.0;   // meaningful in thread 0
    for (int64_t r = blockIdx.x; r < n_con; r += gridDim.x) {
        double sum = 0.0;
        for (int64_t e = ptr[r] + threadIdx.x; e < ptr[r + 1]; e += CON_TPB) sum = fma(val[e], x[col[e]], sum);
        sum = con_block_sum(sum, red);
        if (threadIdx.x == 0) {
            const double ynew = fma(ca, y[r], sum);
            y[r] = ynew;
            q = fma(ynew, ynew, q);
        }
    }
    if (partial && threadIdx.x == 0) partial[blockIdx.x] = q;
}

// x[col[e]] += val[e] * (y[r] * sy)   (SQUARE: x[col[e]] += val[e]^2)
template <bool SQUARE>
__global__ void __launch_bounds__(CON_TPB) k_con_aprod2(int64_t n_con, const int64_t* __restrict__ ptr,
                                                        const int32_t* __restrict__ col,
                                                        const double* __restrict__ val,
                                                        const double* __restrict__ y, double* __restrict__ x,
                                                        const double* __restrict__ sy_p,
                                                        const int* __restrict__ stop) {
    if (stop && *stop) return;
    const double sy = SQUARE ? 1.0 : *sy_p;
    for (int64_t r = blockIdx.x; r < n_con; r += gridDim.x) {
        const double yr = SQUARE ? 1.0 : y[r] * sy;
        for (int64_t e = ptr[r] + threadIdx.x; e < ptr[r + 1]; e += CON_TPB) {
            const double a = val[e];
            const double t = SQUARE ? a * a : a * yr;
            if (t != 0.0) atomicAdd(x + col[e], t);
        }
    }
}

__global__ void k_con_scale(int64_t nnz, const int32_t* __restrict__ col, double* __restrict__ val,
                            const double* __restrict__ p) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < nnz) val[e] *= p[col[e]];
}

// u_hat[m_int + r] = b[m + r]; partial[0] = sum of squares
__global__ void __launch_bounds__(1024) k_con_copy_sumsq(const double* __restrict__ src, double* __restrict__ dst,
                                                         int64_t n_con, double* __restrict__ partial) {
    __shared__ double red[32];
    double q = 0.0;
    for (int64_t r = threadIdx.x; r < n_con; r += 1024) {
        const double t = src[r];
        dst[r] = t;
        q = fma(t, t, q);
    }
    q = wsum(q);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = q;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 32; ++w) t += red[w];
        partial[0] = t;
    }
}

// CTAs of the constraint kernels = partial sums of y^2 they write (CON_GRID_MAX at most)
int con_grid(const gsr_matrix* A) {
    return (int)(A->n_con < CON_GRID_MAX ? A->n_con : CON_GRID_MAX);
}

int launch_con_aprod1(const gsr_matrix* A, const double* x, double* ycon, const double* ca,
                      double* partial, const int* stop, cudaStream_t s) {
    if (A->n_con == 0) return GSR_OK;
    k_con_aprod1<<<con_grid(A), CON_TPB, 0, s>>>(A->n_con, A->con_ptr, A->con_col, A->con_val, x, ycon, ca, partial, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_con_aprod2(const gsr_matrix* A, const double* ycon, double* x, const double* sy,
                      const int* stop, cudaStream_t s) {
    if (A->n_con == 0) return GSR_OK;
    k_con_aprod2<false><<<con_grid(A), CON_TPB, 0, s>>>(A->n_con, A->con_ptr, A->con_col, A->con_val, ycon, x, sy, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_con_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s) {
    if (A->n_con == 0) return GSR_OK;
    k_con_aprod2<true><<<con_grid(A), CON_TPB, 0, s>>>(A->n_con, A->con_ptr, A->con_col, A->con_val, nullptr, q, nullptr, nullptr);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_con_scale(const gsr_matrix* A, const double* p, cudaStream_t s) {
    if (A->n_con == 0 || A->con_nnz == 0) return GSR_OK;
    k_con_scale<<<(unsigned)((A->con_nnz + 255) / 256), 256, 0, s>>>(A->con_nnz, A->con_col, A->con_val, p);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_con_copy_sumsq(const gsr_matrix* A, const double* bcon, double* ucon, double* partial,
                          cudaStream_t s) {
    k_con_copy_sumsq<<<1, 1024, 0, s>>>(bcon, ucon, A->n_con, partial);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

void free_constraints(gsr_matrix* A) {
    dev_free(A, A->con_ptr, (size_t)(A->n_con + 1) * 8);
    dev_free(A, A->con_col, (size_t)A->con_nnz * 4);
    dev_free(A, A->con_val, (size_t)A->con_nnz * 8);
    A->con_ptr = nullptr;
    A->con_col = nullptr;
    A->con_val = nullptr;
    A->n_con = 0;
    A->con_nnz = 0;
}

}  // namespace gsr

using namespace gsr;

extern "C" {

int gsr_matrix_set_constraints(gsr_matrix* A, int64_t n_con, const int64_t* row_ptr_hd,
                               const int32_t* col_hd, const double* val_hd) {
    if (!A || n_con < 0) return GSR_EINVAL;
    if (A->state != 1 || A->p != nullptr || A->ws.st != nullptr) return GSR_ESTATE;   // before precondition / solve
    if (n_con > 0 && !row_ptr_hd) return GSR_EINVAL;
    // on a row shard gsr_matrix_set_comm was told the total number of rows: it must still cover
    // this rank's observations and the constraint rows it is being given now
    if (A->comm && A->m_global < A->dims.n_rows + n_con) return GSR_EINVAL;
    free_constraints(A);
    if (!A->comm) A->m_global = A->dims.n_rows;   // (sharded: gsr_matrix_set_comm was told the total)
    if (n_con == 0) return GSR_OK;
    std::vector<int64_t> ptr((size_t)n_con + 1);
    GSR_CUDA_TRY(cudaMemcpy(ptr.data(), row_ptr_hd, ptr.size() * 8, cudaMemcpyDefault));
    if (ptr[0] != 0) return GSR_EINVAL;
    for (int64_t r = 0; r < n_con; ++r)
        if (ptr[r + 1] < ptr[r]) return GSR_EINVAL;
    const int64_t nnz = ptr[n_con];
    if (nnz > 0 && (!col_hd || !val_hd)) return GSR_EINVAL;
    std::vector<int32_t> col((size_t)nnz);
    if (nnz > 0) GSR_CUDA_TRY(cudaMemcpy(col.data(), col_hd, (size_t)nnz * 4, cudaMemcpyDefault));
    for (int64_t e = 0; e < nnz; ++e)
        if (col[e] < 0 || col[e] >= A->n_cols) return GSR_EINVAL;
    A->n_con = n_con;
    A->con_nnz = nnz;
    int rc = dev_alloc(A, (void**)&A->con_ptr, (size_t)(n_con + 1) * 8);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->con_col, (size_t)nnz * 4);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->con_val, (size_t)nnz * 8);
    if (rc != GSR_OK) {
        free_constraints(A);
        return rc;
    }
    cudaError_t e = cudaMemcpy(A->con_ptr, ptr.data(), ptr.size() * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nnz > 0) e = cudaMemcpy(A->con_col, col.data(), (size_t)nnz * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nnz > 0) e = cudaMemcpy(A->con_val, val_hd, (size_t)nnz * 8, cudaMemcpyDefault);
    if (e != cudaSuccess) {
        cudaGetLastError();
        free_constraints(A);
        return GSR_ECUDA;
    }
    if (!A->comm) A->m_global = A->dims.n_rows + n_con;
    return GSR_OK;
}

}  // extern "C"
