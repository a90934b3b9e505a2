// Matrix ingest (row a0), preconditioner (row a1) and housekeeping of libgsr_b200.
// The operations are defined in include/gsr.h; structure per PAPER.md:73-79.
#include <stdio.h>
#include <string.h>

#include <new>

#include "gsr_internal.h"

namespace gsr {

long long g_launches = 0;

bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

bool is_pinned_host_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeHost;
}

int dev_alloc(gsr_matrix* A, void** p, size_t bytes) {
    *p = nullptr;
    if (bytes == 0) bytes = 8;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        *p = nullptr;
        return e == cudaErrorMemoryAllocation ? GSR_ENOMEM : GSR_ECUDA;
    }
    A->device_bytes += (int64_t)bytes;
    return GSR_OK;
}

// AoS caller form -> tile records.  One thread per row.  Validation sets bits in *err:
// 1 star out of range, 2 star decreasing, 4 att_start out of range, 8 instr_col out of range.
__global__ void k_layout_rows(unsigned char* __restrict__ tiles, int64_t row0, int64_t nrows,
                              const int32_t* __restrict__ star, const int32_t* __restrict__ att,
                              const int32_t* __restrict__ instr, const double* __restrict__ vals,
                              int64_t S, int64_t D, int64_t I, int* __restrict__ err) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nrows) return;
    int64_t row = row0 + r;
    unsigned char* T = tiles + (row / R) * (int64_t)TILE_BYTES;
    int lr = (int)(row % R);
    int e = 0;
    int32_t s = star[r], a = att[r];
    if (s < 0 || s >= S) e |= 1;
    int32_t sprev;
    if (r > 0) sprev = star[r - 1];
    else if (row > 0) {
        const unsigned char* Tp = tiles + ((row - 1) / R) * (int64_t)TILE_BYTES;
        sprev = ((const int32_t*)(Tp + OFF_STAR))[(row - 1) % R];
    } else sprev = 0;
    if (s < sprev) e |= 2;
    if (a < 0 || a > D - 4) e |= 4;
    ((int32_t*)(T + OFF_STAR))[lr] = s;
    ((int32_t*)(T + OFF_ATT))[lr] = a;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        int32_t c = instr[6 * r + j];
        if (c < 0 || c >= I) e |= 8;
        ((int32_t*)(T + OFF_INSTR + j * R * 4))[lr] = c;
    }
#pragma unroll
    for (int k = 0; k < NPAR; ++k) ((double*)(T + k * R * 8))[lr] = vals[NPAR * r + k];
    if (e) atomicOr(err, e);
}

__global__ void k_expand_rows(const unsigned char* __restrict__ tiles, int64_t row0, int64_t nrows,
                              int64_t S, int64_t D, int64_t I, int64_t* __restrict__ cols,
                              double* __restrict__ vals) {
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nrows) return;
    int64_t row = row0 + r;
    const unsigned char* T = tiles + (row / R) * (int64_t)TILE_BYTES;
    int lr = (int)(row % R);
    int64_t s = ((const int32_t*)(T + OFF_STAR))[lr];
    int64_t a = ((const int32_t*)(T + OFF_ATT))[lr];
    const int64_t off_att = 5 * S, off_instr = off_att + 3 * D, off_glob = off_instr + I;
    for (int k = 0; k < NPAR; ++k) {
        int64_t c;
        if (k < 5) c = 5 * s + k;
        else if (k < 17) c = off_att + ((k - 5) / 4) * D + a + (k - 5) % 4;
        else if (k < 23) c = off_instr + ((const int32_t*)(T + OFF_INSTR + (k - 17) * R * 4))[lr];
        else c = off_glob;
        cols[NPAR * r + k] = c;
        vals[NPAR * r + k] = ((const double*)(T + k * R * 8))[lr];
    }
}

// p_j = q_j > 0 ? 1/sqrt(q_j) : 1   (reading A7)
__global__ void k_make_p(double* __restrict__ p, int64_t n) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    double q = p[j];
    p[j] = q > 0.0 ? 1.0 / sqrt(q) : 1.0;
}

// values[i,k] *= p[col(i,k)] in place, one thread per row of a tile.
__global__ void __launch_bounds__(R) k_scale_values(unsigned char* __restrict__ tiles,
                                                    const double* __restrict__ p, int64_t S,
                                                    int64_t D, int64_t I) {
    unsigned char* T = tiles + (int64_t)blockIdx.x * TILE_BYTES;
    const int lr = threadIdx.x;
    const int64_t s = ((const int32_t*)(T + OFF_STAR))[lr];
    const int64_t a = ((const int32_t*)(T + OFF_ATT))[lr];
    const double* pa = p + 5 * s;
    const double* pt = p + 5 * S + a;
    const double* pi = p + 5 * S + 3 * D;
#pragma unroll
    for (int k = 0; k < 5; ++k) ((double*)(T + k * R * 8))[lr] *= pa[k];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax)
#pragma unroll
        for (int j = 0; j < 4; ++j) ((double*)(T + (5 + 4 * ax + j) * R * 8))[lr] *= pt[ax * D + j];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        int32_t c = ((const int32_t*)(T + OFF_INSTR + j * R * 4))[lr];
        ((double*)(T + (17 + j) * R * 8))[lr] *= pi[c];
    }
    ((double*)(T + 23 * R * 8))[lr] *= pi[I];
}

}  // namespace gsr

using namespace gsr;

extern "C" {

const char* gsr_strerror(int code) {
    switch (code) {
        case GSR_OK: return "ok";
        case GSR_EINVAL: return "invalid argument (null pointer, bad dims or index out of range)";
        case GSR_ENOMEM: return "out of device memory";
        case GSR_ECUDA: return "CUDA runtime error";
        case GSR_ESTATE: return "call not legal in this state";
        case GSR_EUNSUPPORTED: return "unsupported device (needs sm_100) or option";
        default: return "unknown gsr status";
    }
}

int64_t gsr_launch_count(void) { return g_launches; }

int gsr_matrix_begin(gsr_matrix** out, const gsr_dims* d, gsr_stream stream) {
    if (!out) return GSR_EINVAL;
    *out = nullptr;
    if (!d) return GSR_EINVAL;
    if (d->n_rows < 0 || d->n_stars < 1 || d->n_dfa < 4 || d->n_instr < 1 || d->n_glob != 1)
        return GSR_EINVAL;
    int64_t n = 5 * d->n_stars + 3 * d->n_dfa + d->n_instr + 1;
    if (n >= (int64_t)1 << 31) return GSR_EINVAL;
    int dev = 0;
    cudaDeviceProp prop;
    GSR_CUDA_TRY(cudaGetDevice(&dev));
    GSR_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return GSR_EUNSUPPORTED;
    gsr_matrix* A = new (std::nothrow) gsr_matrix();
    if (!A) return GSR_ENOMEM;
    memset((void*)A, 0, sizeof(*A));
    new (&A->ws) Workspace();
    A->dims = *d;
    A->n_cols = n;
    A->off_att = 5 * d->n_stars;
    A->off_instr = A->off_att + 3 * d->n_dfa;
    A->off_glob = A->off_instr + d->n_instr;
    A->n_tiles = (d->n_rows + R - 1) / R;
    A->m_pad = A->n_tiles * R;
    A->stream = (cudaStream_t)stream;
    A->sm_count = prop.multiProcessorCount;
    int rc = dev_alloc(A, (void**)&A->tiles, (size_t)A->n_tiles * TILE_BYTES);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->err, sizeof(int));
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->coef_one, 2 * sizeof(double));
    if (rc != GSR_OK) {
        gsr_matrix_destroy(A);
        return rc;
    }
    const double ones[2] = {1.0, 1.0};
    cudaError_t e = cudaMemsetAsync(A->tiles, 0, (size_t)A->n_tiles * TILE_BYTES, A->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A->err, 0, sizeof(int), A->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(A->coef_one, ones, sizeof(ones), cudaMemcpyHostToDevice, A->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(A->stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        gsr_matrix_destroy(A);
        return GSR_ECUDA;
    }
    *out = A;
    return GSR_OK;
}

static int append_device(gsr_matrix* A, int64_t row0, int64_t nrows, const int32_t* star,
                         const int32_t* att, const int32_t* instr, const double* vals) {
    if (nrows == 0) return GSR_OK;
    const int threads = 256;
    const int64_t blocks = (nrows + threads - 1) / threads;
    k_layout_rows<<<(unsigned)blocks, threads, 0, A->stream>>>(A->tiles, row0, nrows, star, att, instr, vals,
                                                               A->dims.n_stars, A->dims.n_dfa,
                                                               A->dims.n_instr, A->err);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int gsr_matrix_append_rows(gsr_matrix* A, int64_t row0, int64_t nrows, const int32_t* star,
                           const int32_t* att, const int32_t* instr, const double* vals) {
    if (!A) return GSR_EINVAL;
    if (A->state != 0) return GSR_ESTATE;
    if (nrows < 0 || row0 != A->rows_appended || row0 + nrows > A->dims.n_rows) return GSR_EINVAL;
    if (nrows == 0) return GSR_OK;
    if (!star || !att || !instr || !vals) return GSR_EINVAL;
    const bool dev = is_device_ptr(star);
    if (dev != is_device_ptr(att) || dev != is_device_ptr(instr) || dev != is_device_ptr(vals))
        return GSR_EINVAL;
    if (dev) {
        GSR_TRY(append_device(A, row0, nrows, star, att, instr, vals));
    } else {
        // host arrays: stage through a bounded device buffer (224 B per row)
        const int64_t chunk = 1 << 20;
        const size_t need = (size_t)(nrows < chunk ? nrows : chunk) * 224;
        if (A->stage_bytes < need) {
            if (A->stage) {
                cudaFree(A->stage);
                A->device_bytes -= (int64_t)A->stage_bytes;
                A->stage = nullptr;
                A->stage_bytes = 0;
            }
            GSR_TRY(dev_alloc(A, &A->stage, need));
            A->stage_bytes = need;
        }
        for (int64_t r0 = 0; r0 < nrows; r0 += chunk) {
            int64_t nr = nrows - r0 < chunk ? nrows - r0 : chunk;
            unsigned char* sb = (unsigned char*)A->stage;
            double* dv = (double*)sb;
            int32_t* ds = (int32_t*)(sb + (size_t)nr * 192);
            int32_t* da = ds + nr;
            int32_t* di = da + nr;
            GSR_CUDA_TRY(cudaMemcpyAsync(dv, vals + 24 * r0, (size_t)nr * 192, cudaMemcpyHostToDevice, A->stream));
            GSR_CUDA_TRY(cudaMemcpyAsync(ds, star + r0, (size_t)nr * 4, cudaMemcpyHostToDevice, A->stream));
            GSR_CUDA_TRY(cudaMemcpyAsync(da, att + r0, (size_t)nr * 4, cudaMemcpyHostToDevice, A->stream));
            GSR_CUDA_TRY(cudaMemcpyAsync(di, instr + 6 * r0, (size_t)nr * 24, cudaMemcpyHostToDevice, A->stream));
            GSR_TRY(append_device(A, row0 + r0, nr, ds, da, di, dv));
            // the staging buffer is reused by the next chunk
            GSR_CUDA_TRY(cudaStreamSynchronize(A->stream));
        }
    }
    A->rows_appended += nrows;
    return GSR_OK;
}

int gsr_matrix_finalize(gsr_matrix* A) {
    if (!A) return GSR_EINVAL;
    if (A->state != 0) return GSR_ESTATE;
    if (A->rows_appended != A->dims.n_rows) return GSR_ESTATE;
    int err = 0;
    GSR_CUDA_TRY(cudaMemcpyAsync(&err, A->err, sizeof(int), cudaMemcpyDeviceToHost, A->stream));
    GSR_CUDA_TRY(cudaStreamSynchronize(A->stream));
    if (A->stage) {
        cudaFree(A->stage);
        A->device_bytes -= (int64_t)A->stage_bytes;
        A->stage = nullptr;
        A->stage_bytes = 0;
    }
    if (err != 0) return GSR_EINVAL;
    A->state = 1;
    return GSR_OK;
}

int gsr_matrix_create(gsr_matrix** out, const gsr_dims* dims, const int32_t* star,
                      const int32_t* att, const int32_t* instr, const double* vals,
                      gsr_stream stream) {
    if (!out) return GSR_EINVAL;
    *out = nullptr;
    if (!dims) return GSR_EINVAL;
    if (dims->n_rows > 0 && (!star || !att || !instr || !vals)) return GSR_EINVAL;
    gsr_matrix* A = nullptr;
    GSR_TRY(gsr_matrix_begin(&A, dims, stream));
    int rc = gsr_matrix_append_rows(A, 0, dims->n_rows, star, att, instr, vals);
    if (rc == GSR_OK) rc = gsr_matrix_finalize(A);
    if (rc != GSR_OK) {
        gsr_matrix_destroy(A);
        return rc;
    }
    *out = A;
    return GSR_OK;
}

int gsr_matrix_destroy(gsr_matrix* A) {
    if (!A) return GSR_OK;
    free_workspace(A);
    cudaFree(A->tiles);
    cudaFree(A->p);
    cudaFree(A->err);
    cudaFree(A->coef_one);
    cudaFree(A->stage);
    cudaGetLastError();
    delete A;
    return GSR_OK;
}

int gsr_matrix_dims(const gsr_matrix* A, gsr_dims* out, int64_t* n_cols) {
    if (!A) return GSR_EINVAL;
    if (out) *out = A->dims;
    if (n_cols) *n_cols = A->n_cols;
    return GSR_OK;
}

int64_t gsr_matrix_device_bytes(const gsr_matrix* A) { return A ? A->device_bytes : 0; }

int gsr_set_option(gsr_matrix* A, int key, int64_t value) {
    if (!A) return GSR_EINVAL;
    switch (key) {
        case GSR_OPT_FORCE_ITNLIM: A->opt_force_itnlim = value != 0; return GSR_OK;
        case GSR_OPT_DETERMINISTIC: A->opt_deterministic = value != 0; return GSR_OK;
        default: return GSR_EINVAL;
    }
}

int gsr_debug_expand_rows(const gsr_matrix* A, int64_t row0, int64_t nrows, int64_t* cols_host,
                          double* vals_host) {
    if (!A || !cols_host || !vals_host) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    if (row0 < 0 || nrows < 0 || row0 + nrows > A->dims.n_rows) return GSR_EINVAL;
    if (nrows == 0) return GSR_OK;
    int64_t* dc = nullptr;
    double* dv = nullptr;
    GSR_CUDA_TRY(cudaMalloc(&dc, (size_t)nrows * NPAR * 8));
    cudaError_t e = cudaMalloc(&dv, (size_t)nrows * NPAR * 8);
    if (e != cudaSuccess) {
        cudaFree(dc);
        cudaGetLastError();
        return GSR_ENOMEM;
    }
    k_expand_rows<<<(unsigned)((nrows + 255) / 256), 256, 0, A->stream>>>(
        A->tiles, row0, nrows, A->dims.n_stars, A->dims.n_dfa, A->dims.n_instr, dc, dv);
    count_launch();
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(cols_host, dc, (size_t)nrows * NPAR * 8, cudaMemcpyDeviceToHost, A->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(vals_host, dv, (size_t)nrows * NPAR * 8, cudaMemcpyDeviceToHost, A->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(A->stream);
    cudaFree(dc);
    cudaFree(dv);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return GSR_ECUDA;
    }
    return GSR_OK;
}

int gsr_precondition(gsr_matrix* A, double* p_out, gsr_stream stream) {
    if (!A) return GSR_EINVAL;
    if (A->state != 1 || A->p != nullptr) return GSR_ESTATE;
    cudaStream_t s = (cudaStream_t)stream;
    GSR_TRY(dev_alloc(A, (void**)&A->p, (size_t)A->n_cols * 8));
    GSR_CUDA_TRY(cudaMemsetAsync(A->p, 0, (size_t)A->n_cols * 8, s));
    GSR_TRY(launch_colsumsq(A, A->p, s));
    k_make_p<<<(unsigned)((A->n_cols + 255) / 256), 256, 0, s>>>(A->p, A->n_cols);
    count_launch();
    if (A->n_tiles > 0) {
        k_scale_values<<<(unsigned)A->n_tiles, R, 0, s>>>(A->tiles, A->p, A->dims.n_stars,
                                                          A->dims.n_dfa, A->dims.n_instr);
        count_launch();
    }
    GSR_CUDA_TRY(cudaGetLastError());
    if (p_out) {
        if (is_device_ptr(p_out)) {
            GSR_CUDA_TRY(cudaMemcpyAsync(p_out, A->p, (size_t)A->n_cols * 8, cudaMemcpyDeviceToDevice, s));
        } else {
            GSR_CUDA_TRY(cudaMemcpyAsync(p_out, A->p, (size_t)A->n_cols * 8, cudaMemcpyDeviceToHost, s));
            GSR_CUDA_TRY(cudaStreamSynchronize(s));
        }
    }
    A->ws.graph_valid = false;
    return GSR_OK;
}

}  // extern "C"
