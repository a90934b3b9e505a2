// LSQR iteration on the device (rows a2, a4, a9-a12): Paige & Saunders 1982 as cited by the
// paper (loop skeleton Algorithm 3), written
// out in DESIGN.md reading C3.  All scalars live in device memory (LsqrState); one iteration
// is a fixed kernel sequence captured in a CUDA graph (row a11).
//
// Deferred normalisation: u is stored unnormalised (u_hat = beta*u); the factor 1/beta is
// folded into aprod2's input and -alpha/beta into aprod1's update, so the m-sized vector is
// read and written exactly once per product.
#include <math.h>
#include <string.h>

#include "gsr_internal.h"

namespace gsr {

constexpr int NB_N = 592;     // CTAs of the n-sized kernels (4 per SM on 148 SMs)
constexpr int TB_N = 256;

__device__ __forceinline__ double block_sum_256(double v, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 0; w < TB_N / 32; ++w) t += red[w];
    }
    return t;  // valid in thread 0
}

// Row-sharded solve (row e): entries below `split` belong to the distributed (astrometric)
// slice, whose sum of squares must still be summed over the ranks, entries from `split` on to
// the replicated slice, counted once.  Without a communicator split = 0 and parta is unused.
__device__ __forceinline__ void write_split_partials(double q, double qa, int64_t split, double* red,
                                                     double* __restrict__ part, double* __restrict__ parta) {
    q = block_sum_256(q, red);
    if (threadIdx.x == 0) part[blockIdx.x] = q;
    if (split > 0) {
        __syncthreads();
        qa = block_sum_256(qa, red);
        if (threadIdx.x == 0) parta[blockIdx.x] = qa;
    }
}

// Deterministic second stage: one CTA sums `np` partials in a fixed order.
__device__ double reduce_partials_1024(const double* __restrict__ part, int64_t np, double* red) {
    double t = 0.0;
    for (int64_t i = threadIdx.x; i < np; i += 1024) t += part[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = t;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = red[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    }
    __syncthreads();
    return r;  // valid in warp 0
}

__device__ __forceinline__ double hyp(double a, double b) { return sqrt(a * a + b * b); }

// u_hat = b gathered into the internal row order (padding rows zero), partial sums of b^2
__global__ void __launch_bounds__(TB_N) k_gather_sumsq(const double* __restrict__ src,
                                                       const uint32_t* __restrict__ perm,
                                                       double* __restrict__ dst, int64_t len_int,
                                                       double* __restrict__ part) {
    __shared__ double red[TB_N / 32];
    double q = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * TB_N + threadIdx.x; i < len_int; i += (int64_t)gridDim.x * TB_N) {
        const uint32_t pe = perm[i];
        double t = pe != PERM_PAD ? src[pe] : 0.0;
        dst[i] = t;
        q = fma(t, t, q);
    }
    q = block_sum_256(q, red);
    if (threadIdx.x == 0) part[blockIdx.x] = q;
}

// dst[perm[i]] = src[i]: an internal-order m-vector back to the caller's row order
__global__ void __launch_bounds__(TB_N) k_scatter_rows(const double* __restrict__ src,
                                                       const uint32_t* __restrict__ perm,
                                                       double* __restrict__ dst, int64_t len_int) {
    for (int64_t i = (int64_t)blockIdx.x * TB_N + threadIdx.x; i < len_int; i += (int64_t)gridDim.x * TB_N) {
        const uint32_t pe = perm[i];
        if (pe != PERM_PAD) dst[pe] = src[i];
    }
}

__global__ void __launch_bounds__(TB_N) k_sumsq(const double* __restrict__ v, int64_t len,
                                                double* __restrict__ part, const int* __restrict__ stop,
                                                int64_t split, double* __restrict__ parta) {
    if (stop && *stop) return;
    __shared__ double red[TB_N / 32];
    double q = 0.0, qa = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * TB_N + threadIdx.x; i < len; i += (int64_t)gridDim.x * TB_N) {
        double t = v[i];
        if (i < split) qa = fma(t, t, qa);
        else q = fma(t, t, q);
    }
    write_split_partials(q, qa, split, red, part, parta);
}

// out[0] = sum of np partials in a fixed order (one CTA); the scalar then crosses the ranks
__global__ void __launch_bounds__(1024) k_sum_partials(const double* __restrict__ part, int64_t np,
                                                       double* __restrict__ out,
                                                       const int* __restrict__ stop) {
    if (stop && *stop) return;
    __shared__ double red[32];
    double ss = reduce_partials_1024(part, np, red);
    if (threadIdx.x == 0) out[0] = ss;
}

// v <- vscale * v   (v = -beta v before aprod2 adds A^T u)
__global__ void __launch_bounds__(TB_N) k_prescale(double* __restrict__ v, int64_t len,
                                                   const LsqrState* __restrict__ st) {
    if (st->stop) return;
    const double c = st->vscale;
    for (int64_t i = (int64_t)blockIdx.x * TB_N + threadIdx.x; i < len; i += (int64_t)gridDim.x * TB_N)
        v[i] = c * v[i];
}

// v <- t * inv_beta + vscale * v  (= A^T u - beta v with t = A^T u_hat from the fused pass) and
// partial sums of the new v squared
__global__ void __launch_bounds__(TB_N) k_vnew(double* __restrict__ v, const double* __restrict__ t,
                                               int64_t len, const LsqrState* __restrict__ st,
                                               double* __restrict__ part, int64_t split,
                                               double* __restrict__ parta) {
    if (st->stop) return;
    __shared__ double red[TB_N / 32];
    const double ib = st->inv_beta, c = st->vscale;
    double q = 0.0, qa = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * TB_N + threadIdx.x; i < len; i += (int64_t)gridDim.x * TB_N) {
        const double vn = fma(t[i], ib, c * v[i]);
        v[i] = vn;
        if (i < split) qa = fma(vn, vn, qa);
        else q = fma(vn, vn, q);
    }
    write_split_partials(q, qa, split, red, part, parta);
}

// fused n-sized update (row a10): v <- v*inv_alpha ; x += t1 w ; w = v + t2 w ; partials of
// the NEW w squared (used as ||w||^2 by the next iteration's ddnorm, reading A10).
// INIT: w = v (first step), x untouched (already zero).
template <bool INIT>
__global__ void __launch_bounds__(TB_N) k_update(double* __restrict__ v, double* __restrict__ w,
                                                 double* __restrict__ x, int64_t len,
                                                 const LsqrState* __restrict__ st,
                                                 double* __restrict__ part_w, double* __restrict__ tz,
                                                 double* __restrict__ var, int64_t split,
                                                 double* __restrict__ part_wa) {
    if (st->stop) return;
    __shared__ double red[TB_N / 32];
    const double ia = st->inv_alpha, t1 = st->t1, t2 = st->t2, ir = st->inv_rho;
    double q = 0.0, qa = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * TB_N + threadIdx.x; i < len; i += (int64_t)gridDim.x * TB_N) {
        double vn = v[i] * ia;
        v[i] = vn;
        double wn;
        if (INIT) {
            wn = vn;
        } else {
            double wo = w[i];
            const double dk = wo * ir;          // var_j += (w_j / rho)^2  (row f1)
            var[i] = fma(dk, dk, var[i]);
            x[i] = fma(t1, wo, x[i]);
            wn = fma(t2, wo, vn);
        }
        w[i] = wn;
        if (tz) tz[i] = 0.0;   // clears the accumulator of the next fused pass
        if (i < split) qa = fma(wn, wn, qa);
        else q = fma(wn, wn, q);
    }
    write_split_partials(q, qa, split, red, part_w, part_wa);
}

// x_out = p (.) z  ("re-multiply the solution by the preconditioning vector")
__global__ void k_finalize_x(const double* __restrict__ z, const double* __restrict__ p,
                             double* __restrict__ out, int64_t len) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < len) out[i] = p ? p[i] * z[i] : z[i];
}

// se_j = p_j * rnorm * sqrt(var_j / dof)   (row f1; Paige & Saunders' standard errors, scaled
// back by p like the solution)
__global__ void k_standard_errors(const double* __restrict__ var, const double* __restrict__ p,
                                  double rnorm, double dof, double* __restrict__ out, int64_t len) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= len) return;
    const double e = rnorm * sqrt(var[i] / dof);
    out[i] = p ? p[i] * e : e;
}

// ---- scalar kernels (rows a4, a9): one CTA, deterministic second-stage sums, then one
// thread runs the recurrences of reading C3 ------------------------------------------------

// beta_1 = ||b||
__global__ void __launch_bounds__(1024) k_scalar_init1(LsqrState* __restrict__ st,
                                                       const double* __restrict__ part_u, int64_t np,
                                                       double* __restrict__ sum_out) {
    __shared__ double red[32];
    double ss = reduce_partials_1024(part_u, np, red);
    if (threadIdx.x != 0) return;
    if (sum_out) *sum_out = ss;   // ||b||^2: the range of the initial aprod2's fixed-point pass
    double beta = sqrt(ss);
    st->beta = beta;
    st->bnorm = beta;
    st->rnorm = beta;
    st->beta_pos = beta > 0.0;
    if (beta == 0.0) {          // x = 0 is the exact solution
        st->stop = 1;
        st->istop = 0;
        st->inv_beta = 0.0;
    } else {
        st->inv_beta = 1.0 / beta;
        st->det_e = ilogb(beta) + 2;   // deterministic init pass: u_hat = b, ||u_hat|| = beta_1 < 2^det_e
    }
}

// alpha_1 = ||A^T u_1||
__global__ void __launch_bounds__(1024) k_scalar_init2(LsqrState* __restrict__ st,
                                                       const double* __restrict__ part_v, int64_t np,
                                                       const double* __restrict__ extra) {
    if (st->stop) return;
    __shared__ double red[32];
    double ss = reduce_partials_1024(part_v, np, red);
    if (extra) ss += extra[0];   // distributed slice, already summed over the ranks
    if (threadIdx.x != 0) return;
    double alpha = sqrt(ss);
    st->alpha = alpha;
    if (alpha == 0.0) {
        st->stop = 1;
        st->istop = 0;
        st->inv_alpha = 1.0;
        return;
    }
    st->inv_alpha = 1.0 / alpha;
    st->rhobar = alpha;
    st->phibar = st->beta;
    st->arnorm = alpha * st->beta;
    st->ca = -alpha / st->beta;
    // range of the first fused pass (deterministic mode): ||u_hat_1|| = beta_2 <= ||A||_2
    st->det_max = alpha;
    st->det_e = min(ilogb(alpha) + 8, st->det_cap);
}

// beta_{k+1} = ||A v_k - alpha_k u_k||, anorm update
// (sum_out, if given, receives sum u_hat^2: the fixed-point scale of the instrumental pass)
__global__ void __launch_bounds__(1024) k_scalar_beta(LsqrState* __restrict__ st,
                                                      const double* __restrict__ part_u, int64_t np,
                                                      double* __restrict__ sum_out) {
    if (st->stop) return;
    __shared__ double red[32];
    double ss = reduce_partials_1024(part_u, np, red);
    if (threadIdx.x != 0) return;
    if (sum_out) *sum_out = ss;
    st->itn += 1;
    double beta = sqrt(ss);
    st->beta = beta;
    if (st->det && !(beta < scalbn(1.0, st->det_e))) {   // the pass left its fixed-point range
        st->det_fail = 1;
        st->stop = 1;
        return;
    }
    if (beta > st->det_max) st->det_max = beta;
    if (beta > 0.0) {
        st->beta_pos = 1;
        st->anorm = hyp(hyp(st->anorm, st->alpha), beta);   // uses the OLD alpha
        if (st->damp > 0.0) st->anorm = hyp(st->anorm, st->damp);
        st->inv_beta = 1.0 / beta;
        st->vscale = -beta;
    } else {
        st->beta_pos = 0;
        st->inv_beta = 0.0;
        st->vscale = 1.0;
    }
}

// alpha_{k+1}, plane rotations, norms, stopping rules
__global__ void __launch_bounds__(1024) k_scalar_main(LsqrState* __restrict__ st,
                                                      const double* __restrict__ part_v,
                                                      const double* __restrict__ part_w, int64_t np,
                                                      const double* __restrict__ extra) {
    if (st->stop) return;
    __shared__ double red[32];
    double ssv = reduce_partials_1024(part_v, np, red);
    double ssw = reduce_partials_1024(part_w, np, red);
    if (extra) {                 // distributed slices, already summed over the ranks
        ssv += extra[0];
        ssw += extra[1];
    }
    if (threadIdx.x != 0) return;
    double alpha = st->alpha;
    const double beta = st->beta;
    if (st->beta_pos) {
        alpha = sqrt(ssv);
        st->inv_alpha = alpha > 0.0 ? 1.0 / alpha : 1.0;
    } else {
        st->inv_alpha = 1.0;
    }
    st->alpha = alpha;
    // plane rotation eliminating the damping parameter (row f4; only when damp > 0)
    double rhobar1 = st->rhobar, psi = 0.0;
    if (st->damp > 0.0) {
        rhobar1 = hyp(st->rhobar, st->damp);
        const double cs1 = st->rhobar / rhobar1, sn1 = st->damp / rhobar1;
        psi = sn1 * st->phibar;
        st->phibar = cs1 * st->phibar;
    }
    // plane rotation eliminating beta
    const double rho = hyp(rhobar1, beta);
    const double cs = rhobar1 / rho, sn = beta / rho;
    const double theta = sn * alpha;
    st->rhobar = -cs * alpha;
    const double phi = cs * st->phibar;
    st->phibar = sn * st->phibar;
    const double tau = sn * phi;
    st->t1 = phi / rho;
    st->t2 = -theta / rho;
    st->inv_rho = 1.0 / rho;
    st->ddnorm = st->ddnorm + ssw / (rho * rho);
    // second rotation: ||x|| estimate
    const double delta = st->sn2 * rho;
    const double gambar = -st->cs2 * rho;
    const double rhs = phi - delta * st->z;
    const double zbar = rhs / gambar;
    const double xnorm = sqrt(st->xxnorm + zbar * zbar);
    const double gamma = hyp(gambar, theta);
    st->cs2 = gambar / gamma;
    st->sn2 = theta / gamma;
    st->z = rhs / gamma;
    st->xxnorm = st->xxnorm + st->z * st->z;
    // norms and stopping tests
    const double anorm = st->anorm, bnorm = st->bnorm;
    const double acond = anorm * sqrt(st->ddnorm);
    st->res2 = st->res2 + psi * psi;
    const double rnorm = st->damp > 0.0 ? sqrt(st->phibar * st->phibar + st->res2) : st->phibar;
    const double arnorm = alpha * fabs(tau);
    st->acond = acond;
    st->rnorm = rnorm;
    st->arnorm = arnorm;
    st->xnorm = xnorm;
    const double test1 = rnorm / bnorm;
    const double test2 = (anorm * rnorm > 0.0) ? arnorm / (anorm * rnorm) : INFINITY;
    const double test3 = 1.0 / acond;
    const double t1c = test1 / (1.0 + anorm * xnorm / bnorm);
    const double rtol = st->btol + st->atol * anorm * xnorm / bnorm;
    int nat = 0;
    if (1.0 + test3 <= 1.0) nat = 6;
    if (1.0 + test2 <= 1.0) nat = 5;
    if (1.0 + t1c <= 1.0) nat = 4;
    if (test3 <= st->ctol) nat = 3;
    if (test2 <= st->atol) nat = 2;
    if (test1 <= rtol) nat = 1;
    if (nat != 0 && st->istop_nat == 0) {
        st->istop_nat = nat;
        st->itn_nat = st->itn;
    }
    int istop = 0;
    if (st->itn >= st->itnlim) istop = 7;
    if (!st->force && nat != 0) istop = nat;
    st->istop = istop;
    // coefficient of the next aprod1: u_hat <- A v - (alpha/beta) u_hat
    st->ca = st->beta_pos ? -alpha / beta : 0.0;
    // deterministic mode: range of the next fused pass.  beta_{k+2} <= ||A||_2, of which the
    // largest alpha / beta seen so far is a close lower estimate: 2^7 of headroom above it,
    // never more than the rigorous cap 2 ||A||_F; k_scalar_beta checks the range afterwards.
    if (alpha > st->det_max) st->det_max = alpha;
    st->det_e = st->det_max > 0.0 ? min(ilogb(st->det_max) + 8, st->det_cap) : st->det_cap;
    // The update kernel of THIS iteration must still run; it checks `stop` first, so the
    // flag is raised by k_raise_stop after it.
}

__global__ void k_raise_stop(LsqrState* __restrict__ st) {
    if (st->istop != 0) st->stop = 1;
}

// Loop condition of the WHILE graph (row a11): run the body again unless the stop flag is up.
// (It is also the body's k_raise_stop: one node less on the critical path of a small system.)
__global__ void k_loop_cond(LsqrState* __restrict__ st, cudaGraphConditionalHandle h) {
    if (st->istop != 0) st->stop = 1;
    cudaGraphSetConditional(h, st->stop ? 0u : 1u);
}

// ---- host side ----------------------------------------------------------------------------

int ensure_workspace(gsr_matrix* A) {
    Workspace& W = A->ws;
    if (W.st) return GSR_OK;
    const size_t n8 = (size_t)A->n_cols * 8;
    int64_t npu = A->n_units > NB_N ? A->n_units : NB_N;
    GSR_TRY(dev_alloc(A, (void**)&W.u, (size_t)(A->m_int + A->n_con) * 8));   // constraint rows at the end
    GSR_TRY(dev_alloc(A, (void**)&W.v, n8));
    GSR_TRY(dev_alloc(A, (void**)&W.w, n8));
    GSR_TRY(dev_alloc(A, (void**)&W.x, n8));
    GSR_TRY(dev_alloc(A, (void**)&W.t, n8 + 16));   // t[n]: local sum of u_hat^2 (sharded solve)
    GSR_TRY(dev_alloc(A, (void**)&W.var, n8));
    GSR_TRY(dev_alloc(A, (void**)&W.part_u, (size_t)(npu + CON_GRID_MAX + 1) * 8));   // + slots of the constraint rows
    GSR_TRY(dev_alloc(A, (void**)&W.part_v, NB_N * 8));
    GSR_TRY(dev_alloc(A, (void**)&W.part_w, NB_N * 8));
    GSR_TRY(dev_alloc(A, (void**)&W.part_va, NB_N * 8));
    GSR_TRY(dev_alloc(A, (void**)&W.part_wa, NB_N * 8));
    GSR_TRY(dev_alloc(A, (void**)&W.red, 4 * 8));
    GSR_TRY(dev_alloc(A, (void**)&W.st, sizeof(LsqrState)));
    GSR_CUDA_TRY(cudaMemset(W.u, 0, (size_t)(A->m_int + A->n_con) * 8));
    GSR_CUDA_TRY(cudaMemset(W.st, 0, sizeof(LsqrState)));
    GSR_CUDA_TRY(cudaMemset(W.red, 0, 4 * 8));
    GSR_CUDA_TRY(cudaMallocHost((void**)&W.stop_host, 64));
    return GSR_OK;
}

void free_workspace(gsr_matrix* A) {
    Workspace& W = A->ws;
    if (W.graph) cudaGraphExecDestroy(W.graph);
    if (W.wgraph) cudaGraphExecDestroy(W.wgraph);
    cudaFree(W.u); cudaFree(W.v); cudaFree(W.w); cudaFree(W.x); cudaFree(W.t); cudaFree(W.var);
    cudaFree(W.part_u); cudaFree(W.part_v); cudaFree(W.part_w);
    cudaFree(W.part_va); cudaFree(W.part_wa); cudaFree(W.red);
    cudaFree(W.stage_m); cudaFree(W.stage_n); cudaFree(W.st);
    if (W.stop_host) cudaFreeHost(W.stop_host);
    if (W.ev0) cudaEventDestroy(W.ev0);
    if (W.ev1) cudaEventDestroy(W.ev1);
    cudaGetLastError();
    W = Workspace();
}

// One LSQR iteration as a fixed kernel sequence (row a11).  Every kernel reads its
// coefficients from LsqrState and returns at once when st->stop is set.
// Fused form (default): the matrix is read once -- k_fused produces u_hat and t = A^T u_hat
// together, k_aprod2_instr adds the instrumental block of t, k_vnew forms v = t/beta - beta v.
// Two-pass form (GSR_OPT_FUSED = 0): aprod1, then aprod2 on the pre-scaled v.
static int kernels_per_iteration(const gsr_matrix* A) {
    return (A->opt_two_pass ? (aprod2_is_split(A) || aprod2_fixed_split(A) ? 9 : 8) : (A->comm ? 10 : 7)) + (A->n_con > 0 ? 2 : 0) +
           (A->opt_deterministic ? 1 : 0);
}

static int enqueue_iteration(gsr_matrix* A, cudaStream_t s, const cudaGraphConditionalHandle* loop = nullptr) {
    Workspace& W = A->ws;
    const int64_t n = A->n_cols;
    const int64_t split = A->comm ? A->off_att : 0;   // sharded: [0, split) distributed slice
    const int ncp = con_grid(A);                      // more partials of u_hat^2 (constraint rows)
    if (A->opt_two_pass) {
        // bidiagonalisation, first half: u_hat <- A v - (alpha/beta) u_hat ; partials of u_hat^2
        GSR_TRY(launch_aprod1(A, W.v, W.u, &W.st->ca, W.part_u, &W.st->stop, nullptr, s));
        GSR_TRY(launch_con_aprod1(A, W.v, W.u + A->m_int, &W.st->ca, W.part_u + A->n_units, &W.st->stop, s));
        k_scalar_beta<<<1, 1024, 0, s>>>(W.st, W.part_u, A->n_units + ncp, W.red + 3);
        // second half: v <- A^T (u_hat/beta) - beta v
        k_prescale<<<NB_N, TB_N, 0, s>>>(W.v, n, W.st);
        GSR_TRY(launch_aprod2(A, W.u, W.v, &W.st->inv_beta, &W.st->stop, nullptr, s, W.red + 3));
        GSR_TRY(launch_con_aprod2(A, W.u + A->m_int, W.v, &W.st->inv_beta, &W.st->stop, s));
        k_sumsq<<<NB_N, TB_N, 0, s>>>(W.v, n, W.part_v, &W.st->stop, 0, nullptr);
        k_scalar_main<<<1, 1024, 0, s>>>(W.st, W.part_v, W.part_w, NB_N, nullptr);
        k_update<false><<<NB_N, TB_N, 0, s>>>(W.v, W.w, W.x, n, W.st, W.part_w, nullptr, W.var, 0, nullptr);
    } else if (A->so.on) {
        // out-of-core (row f4(iii)): k_fused and the instrumental pass run back to back on every
        // view while its tiles are on the device -- the host part crosses the bus once
        GSR_TRY(launch_fused_streamed(A, W.v, W.u, &W.st->ca, W.part_u, W.t, &W.st->stop, s));
        GSR_TRY(launch_con_aprod1(A, W.v, W.u + A->m_int, &W.st->ca, W.part_u + A->n_units, &W.st->stop, s));
        GSR_TRY(launch_con_aprod2(A, W.u + A->m_int, W.t, A->coef_one, &W.st->stop, s));
        k_scalar_beta<<<1, 1024, 0, s>>>(W.st, W.part_u, A->n_units + ncp, W.red + 3);
        k_vnew<<<NB_N, TB_N, 0, s>>>(W.v, W.t, n, W.st, W.part_v, 0, nullptr);
        k_scalar_main<<<1, 1024, 0, s>>>(W.st, W.part_v, W.part_w, NB_N, nullptr);
        k_update<false><<<NB_N, TB_N, 0, s>>>(W.v, W.w, W.x, n, W.st, W.part_w, W.t, W.var, 0, nullptr);
    } else if (!A->comm) {
        const int det = A->opt_deterministic;
        GSR_TRY(launch_fused(A, W.v, W.u, &W.st->ca, W.part_u, W.t, &W.st->stop, det ? &W.st->det_e : nullptr, s));
        // constraint rows (row f3): same two steps on the CSR block, u_hat[m_int ..]
        GSR_TRY(launch_con_aprod1(A, W.v, W.u + A->m_int, &W.st->ca, W.part_u + A->n_units, &W.st->stop, s));
        GSR_TRY(launch_con_aprod2(A, W.u + A->m_int, W.t, A->coef_one, &W.st->stop, s));
        // beta (and sum u_hat^2 for the fixed-point scale of the instrumental pass) in one kernel
        k_scalar_beta<<<1, 1024, 0, s>>>(W.st, W.part_u, A->n_units + ncp, W.red + 3);
        GSR_TRY(launch_aprod2_instr(A, W.u, W.t, W.red + 3, &W.st->stop, det, s));
        if (det) GSR_TRY(launch_det_finish(A, W.t, &W.st->det_e, W.red + 3, &W.st->stop, s));
        k_vnew<<<NB_N, TB_N, 0, s>>>(W.v, W.t, n, W.st, W.part_v, 0, nullptr);
        k_scalar_main<<<1, 1024, 0, s>>>(W.st, W.part_v, W.part_w, NB_N, nullptr);
        k_update<false><<<NB_N, TB_N, 0, s>>>(W.v, W.w, W.x, n, W.st, W.part_w, W.t, W.var, 0, nullptr);
    } else {
        // row-sharded: the same sequence with the paper's two reductions (Alg. 3 lines 12, 16)
        // as NCCL all-reduces inside the graph.  #1: replicated slice of t = A^T u_hat, with the
        // local sum of u_hat^2 riding in t[n]; #2: the distributed parts of ||v||^2 and ||w||^2.
        // Constraint rows belong to the rank that was given them (local column numbering): their
        // part of u_hat^2 and of t joins the local sums before the all-reduce.
        GSR_TRY(launch_fused(A, W.v, W.u, &W.st->ca, W.part_u, W.t, &W.st->stop, nullptr, s));
        GSR_TRY(launch_con_aprod1(A, W.v, W.u + A->m_int, &W.st->ca, W.part_u + A->n_units, &W.st->stop, s));
        GSR_TRY(launch_con_aprod2(A, W.u + A->m_int, W.t, A->coef_one, &W.st->stop, s));
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_u, A->n_units + ncp, W.t + n, &W.st->stop);
        GSR_TRY(launch_aprod2_instr(A, W.u, W.t, W.t + n, &W.st->stop, 0, s));   // local ||u_hat||^2
        GSR_TRY(comm_allreduce_sum(A->comm, W.t + split, (size_t)(n - split + 1), s));
        k_scalar_beta<<<1, 1024, 0, s>>>(W.st, W.t + n, 1, nullptr);
        k_vnew<<<NB_N, TB_N, 0, s>>>(W.v, W.t, n, W.st, W.part_v, split, W.part_va);
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_va, NB_N, W.red, &W.st->stop);
        GSR_TRY(comm_allreduce_sum(A->comm, W.red, 2, s));      // red[1]: from the last k_update
        k_scalar_main<<<1, 1024, 0, s>>>(W.st, W.part_v, W.part_w, NB_N, W.red);
        k_update<false><<<NB_N, TB_N, 0, s>>>(W.v, W.w, W.x, n, W.st, W.part_w, W.t, W.var, split, W.part_wa);
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_wa, NB_N, W.red + 1, &W.st->stop);
    }
    if (loop) k_loop_cond<<<1, 1, 0, s>>>(W.st, *loop);   // body of the WHILE graph
    else k_raise_stop<<<1, 1, 0, s>>>(W.st);
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

static int build_graph(gsr_matrix* A, cudaStream_t s) {
    Workspace& W = A->ws;
    // everything enqueue_iteration() decides at capture time is part of the key: the iteration
    // form, the communicator, the constraint rows, and the variant of the instrumental pass
    // (fixed point needs a scaled matrix and GSR_OPT_FIXED_POINT)
    const int key = (A->opt_two_pass ? 1 : 0) | (A->p != nullptr ? 2 : 0) | (A->opt_no_fixed ? 4 : 0) |
                    (A->n_con > 0 ? 8 : 0) | (A->opt_deterministic ? 16 : 0) | (aprod2_is_split(A) ? 32 : 0) |
                    (A->opt_while ? 64 : 0);
    if (W.graph_valid && W.graph_stream == s && W.graph_key == key && W.graph_comm == (void*)A->comm &&
        W.graph_ncon == A->n_con)
        return GSR_OK;
    if (W.graph) {
        cudaGraphExecDestroy(W.graph);
        W.graph = nullptr;
    }
    cudaStream_t cs = s;
    bool own = false;
    if (s == nullptr || s == cudaStreamLegacy) {   // the legacy stream cannot be captured
        GSR_CUDA_TRY(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
        own = true;
    }
    cudaGraph_t g = nullptr;
    long long before = g_launches;
    cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    int rc = GSR_OK;
    if (e == cudaSuccess) {
        rc = enqueue_iteration(A, cs);
        e = cudaStreamEndCapture(cs, &g);
    }
    g_launches = before;   // capture issues no launches
    if (own) cudaStreamDestroy(cs);
    if (e != cudaSuccess || rc != GSR_OK || !g) {
        cudaGetLastError();
        if (g) cudaGraphDestroy(g);
        return rc != GSR_OK ? rc : GSR_ECUDA;
    }
    e = cudaGraphInstantiate(&W.graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) {
        cudaGetLastError();
        W.graph = nullptr;
        return GSR_ECUDA;
    }
    W.graph_valid = true;
    W.graph_stream = s;
    W.graph_key = key;
    W.graph_ncon = A->n_con;
    W.graph_comm = (void*)A->comm;
    W.graph_builds += 1;
    // The whole loop as ONE graph: a conditional WHILE node whose body is the same iteration with
    // k_loop_cond in the place of k_raise_stop.  One launch per solve, the stop decision never leaves the device.  Not with
    // a communicator (NCCL kernels stay outside conditional bodies).  If the driver refuses any
    // step the per-iteration graph above is what runs (gsr_debug_while_graph tells which).  Built
    // only when GSR_OPT_WHILE_GRAPH asks for it (the option is part of the cache key).
    if (W.wgraph) {
        cudaGraphExecDestroy(W.wgraph);
        W.wgraph = nullptr;
    }
    W.wgraph_tried = true;
    if (!A->comm && A->opt_while) {
        cudaStream_t ws = nullptr;
        cudaGraph_t wg = nullptr;
        bool ok = cudaStreamCreateWithFlags(&ws, cudaStreamNonBlocking) == cudaSuccess;
        ok = ok && cudaGraphCreate(&wg, 0) == cudaSuccess;
        cudaGraphConditionalHandle ch;
        ok = ok && cudaGraphConditionalHandleCreate(&ch, wg, 1, cudaGraphCondAssignDefault) == cudaSuccess;
        cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
        cudaGraphNode_t node;
        if (ok) {
            np.conditional.handle = ch;
            np.conditional.type = cudaGraphCondTypeWhile;
            np.conditional.size = 1;
            ok = cudaGraphAddNode(&node, wg, nullptr, 0, &np) == cudaSuccess;
        }
        if (ok) {
            cudaGraph_t body = np.conditional.phGraph_out[0];
            before = g_launches;
            ok = cudaStreamBeginCaptureToGraph(ws, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
            if (ok) {
                const int rcw = enqueue_iteration(A, ws, &ch);
                cudaGraph_t got = nullptr;
                ok = cudaStreamEndCapture(ws, &got) == cudaSuccess && rcw == GSR_OK;
            }
            g_launches = before;
        }
        ok = ok && cudaGraphInstantiate(&W.wgraph, wg, 0) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();
            W.wgraph = nullptr;
        }
        if (wg) cudaGraphDestroy(wg);
        if (ws) cudaStreamDestroy(ws);
    }
    return GSR_OK;
}

}  // namespace gsr

using namespace gsr;

extern "C" {

int gsr_lsqr_solve(gsr_matrix* A, const double* b_hd, double* x_hd, int64_t itnlim, double atol,
                   double btol, double conlim, gsr_lsqr_result* result, gsr_stream stream) {
    if (!A || !x_hd || !result || (!b_hd && A->dims.n_rows > 0) || itnlim < 1) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    cudaStream_t s = (cudaStream_t)stream;
    Workspace& W = A->ws;
    GSR_TRY(ensure_workspace(A));
    const int64_t m = A->dims.n_rows + A->n_con, n = A->n_cols;   // b: observations then constraints
    memset(result, 0, sizeof(*result));
    if (A->so.on && (A->comm || A->opt_deterministic)) return GSR_EUNSUPPORTED;
    // deterministic mode: fused iteration on a column-scaled matrix (the range bound of its
    // fixed-point sums needs unit column norms), no constraint rows, one GPU
    if (A->opt_deterministic && (!A->p || A->opt_two_pass || A->comm || A->n_con > 0 || A->damp > 0.0))
        return GSR_EUNSUPPORTED;

    // b -> device
    const double* b_dev = b_hd;
    if (m > 0 && !is_device_ptr(b_hd)) {
        if (!W.stage_m) GSR_TRY(dev_alloc(A, (void**)&W.stage_m, (size_t)m * 8));
        GSR_CUDA_TRY(cudaMemcpyAsync(W.stage_m, b_hd, (size_t)m * 8, cudaMemcpyHostToDevice, s));
        b_dev = W.stage_m;
    }
    // state
    LsqrState h;
    memset(&h, 0, sizeof(h));
    h.cs2 = -1.0;
    h.atol = atol;
    h.btol = btol;
    h.ctol = conlim > 0.0 ? 1.0 / conlim : 0.0;
    h.itnlim = itnlim;
    h.force = A->opt_force_itnlim;
    h.damp = A->damp;
    h.inv_alpha = 1.0;
    h.det = A->opt_deterministic;
    h.det_cap = ilogb(2.0 * sqrt((double)n)) + 1;   // ||A'||_2 <= ||A'||_F <= sqrt(n): unit columns
    GSR_CUDA_TRY(cudaMemcpyAsync(W.st, &h, sizeof(h), cudaMemcpyHostToDevice, s));
    GSR_CUDA_TRY(cudaMemsetAsync(W.v, 0, (size_t)n * 8, s));
    GSR_CUDA_TRY(cudaMemsetAsync(W.x, 0, (size_t)n * 8, s));
    GSR_CUDA_TRY(cudaMemsetAsync(W.var, 0, (size_t)n * 8, s));
    W.solved = false;
    // initialisation (row a2): u_hat = b, beta_1, v = A^T u, alpha_1, w = v
    if (A->comm && A->opt_two_pass) return GSR_EUNSUPPORTED;
    const int64_t split = A->comm ? A->off_att : 0;
    k_gather_sumsq<<<NB_N, TB_N, 0, s>>>(b_dev, A->perm, W.u, A->m_int, W.part_u);
    if (A->comm) {   // ||b||^2 over all row shards (each with the constraint rows it owns)
        if (A->n_con > 0)
            GSR_TRY(launch_con_copy_sumsq(A, b_dev + A->dims.n_rows, W.u + A->m_int, W.part_u + NB_N, s));
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_u, NB_N + (A->n_con > 0 ? 1 : 0), W.red + 2, nullptr);
        GSR_TRY(comm_allreduce_sum(A->comm, W.red + 2, 1, s));
        k_scalar_init1<<<1, 1024, 0, s>>>(W.st, W.red + 2, 1, nullptr);
        count_launch();
    } else {
        if (A->n_con > 0)
            GSR_TRY(launch_con_copy_sumsq(A, b_dev + A->dims.n_rows, W.u + A->m_int, W.part_u + NB_N, s));
        k_scalar_init1<<<1, 1024, 0, s>>>(W.st, W.part_u, NB_N + (A->n_con > 0 ? 1 : 0), W.red + 3);
    }
    count_launch(2);
    if (A->opt_deterministic) {
        // v = A^T u_hat / beta_1 through the fused kernels: with v = 0 and ca = 1 the pass leaves
        // u_hat = b as it is and accumulates t = A^T b in fixed point (range: ||b|| = beta_1)
        GSR_CUDA_TRY(cudaMemsetAsync(W.t, 0, (size_t)n * 8, s));
        GSR_TRY(launch_fused(A, W.v, W.u, A->coef_one, W.part_u, W.t, &W.st->stop, &W.st->det_e, s));
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_u, A->n_units, W.red + 3, &W.st->stop);
        GSR_TRY(launch_aprod2_instr(A, W.u, W.t, W.red + 3, &W.st->stop, 1, s));
        GSR_TRY(launch_det_finish(A, W.t, &W.st->det_e, W.red + 3, &W.st->stop, s));
        k_vnew<<<NB_N, TB_N, 0, s>>>(W.v, W.t, n, W.st, W.part_v, 0, nullptr);   // v = t / beta_1
        count_launch(2);
    } else {
    // (single GPU: ||b||^2 is known, the instrumental block takes the fixed-point pass)
    GSR_TRY(launch_aprod2(A, W.u, W.v, &W.st->inv_beta, &W.st->stop, nullptr, s, A->comm ? nullptr : W.red + 3));
    GSR_TRY(launch_con_aprod2(A, W.u + A->m_int, W.v, &W.st->inv_beta, &W.st->stop, s));
    if (A->comm)     // replicated slice of v = A^T u: sum of the shards' contributions
        GSR_TRY(comm_allreduce_sum(A->comm, W.v + split, (size_t)(n - split), s));
    k_sumsq<<<NB_N, TB_N, 0, s>>>(W.v, n, W.part_v, &W.st->stop, split, W.part_va);
    if (A->comm) {
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_va, NB_N, W.red, &W.st->stop);
        GSR_TRY(comm_allreduce_sum(A->comm, W.red, 1, s));
        count_launch();
    }
    }
    k_scalar_init2<<<1, 1024, 0, s>>>(W.st, W.part_v, NB_N, A->comm ? W.red : nullptr);
    k_update<true><<<NB_N, TB_N, 0, s>>>(W.v, W.w, W.x, n, W.st, W.part_w, nullptr, nullptr, split, W.part_wa);
    if (A->comm) {
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_wa, NB_N, W.red + 1, &W.st->stop);
        count_launch();
    }
    GSR_CUDA_TRY(cudaMemsetAsync(W.t, 0, (size_t)n * 8, s));
    count_launch(3);
    GSR_CUDA_TRY(cudaGetLastError());

    // the loop: graph launches; the stop flag is polled from pinned memory between batches
    const bool use_graph = !A->so.on;   // streamed: two streams and copies per pass, enqueued by the host
    if (use_graph) GSR_TRY(build_graph(A, s));
    if (!W.ev0) {
        GSR_CUDA_TRY(cudaEventCreate(&W.ev0));
        GSR_CUDA_TRY(cudaEventCreate(&W.ev1));
    }
    GSR_CUDA_TRY(cudaEventRecord(W.ev0, s));   // device time of the iterations alone (bench.py)
    // (fixed-count mode never stops early; with a communicator every launch that follows the stop
    // still runs its two all-reduces, so the stop flag is polled more often there)
    // Streamed handles: nothing in an iteration needs a host value (every kernel checks the stop
    // flag), so fixed-count mode enqueues 8 iterations per poll and the copy stream never waits for
    // the host; in standard mode a launch that follows the stop would still move the whole host
    // part over the bus, so the flag is polled after every iteration there.
    const int64_t batch = !use_graph ? (A->opt_force_itnlim ? 8 : 1) : A->opt_force_itnlim ? 256 : A->comm ? 8 : 32;
    int64_t launched = 0;
    W.last_loop_while = use_graph && W.wgraph != nullptr && A->opt_while;
    if (W.last_loop_while) {
        // every iteration up to the stop (itn >= itnlim raises it too) in one launch
        GSR_CUDA_TRY(cudaGraphLaunch(W.wgraph, s));
        launched = itnlim;
    }
    while (launched < itnlim) {
        int64_t nb = itnlim - launched < batch ? itnlim - launched : batch;
        if (use_graph) {
            for (int64_t i = 0; i < nb; ++i) GSR_CUDA_TRY(cudaGraphLaunch(W.graph, s));
            count_launch(nb * kernels_per_iteration(A));
        } else {
            for (int64_t i = 0; i < nb; ++i) {
                GSR_TRY(enqueue_iteration(A, s));   // (its launchers count their own launches)
                count_launch(5);
            }
        }
        launched += nb;
        GSR_CUDA_TRY(cudaMemcpyAsync(W.stop_host, &W.st->stop, sizeof(int), cudaMemcpyDeviceToHost, s));
        GSR_CUDA_TRY(cudaStreamSynchronize(s));
        if (*W.stop_host) break;
    }
    GSR_CUDA_TRY(cudaEventRecord(W.ev1, s));
    // finalisation (row a12)
    const bool x_dev = is_device_ptr(x_hd);
    double* xo = x_hd;
    if (!x_dev) {
        if (!W.stage_n) GSR_TRY(dev_alloc(A, (void**)&W.stage_n, (size_t)n * 8));
        xo = W.stage_n;
    }
    k_finalize_x<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(W.x, A->p, xo, n);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    if (!x_dev) GSR_CUDA_TRY(cudaMemcpyAsync(x_hd, xo, (size_t)n * 8, cudaMemcpyDeviceToHost, s));
    GSR_CUDA_TRY(cudaMemcpyAsync(&h, W.st, sizeof(h), cudaMemcpyDeviceToHost, s));
    GSR_CUDA_TRY(cudaStreamSynchronize(s));
    if (W.last_loop_while) count_launch(h.itn * kernels_per_iteration(A));
    if (h.det_fail) return GSR_ERANGE;
    result->istop = h.istop;
    result->istop_natural = h.istop_nat;
    result->itn = h.itn;
    result->itn_natural = h.itn_nat;
    result->rnorm = h.rnorm;
    result->arnorm = h.arnorm;
    result->anorm = h.anorm;
    result->acond = h.acond;
    result->xnorm = h.xnorm;
    result->bnorm = h.bnorm;
    if (result->istop_natural == 0 && h.istop != 7) result->istop_natural = h.istop;
    W.solved = true;
    W.last_rnorm = h.rnorm;
    float loop_ms = 0.f;
    if (cudaEventElapsedTime(&loop_ms, W.ev0, W.ev1) != cudaSuccess) cudaGetLastError();
    W.last_loop_ms = loop_ms;
    return GSR_OK;
}

int gsr_lsqr_set_damp(gsr_matrix* A, double damp) {
    if (!A || !(damp >= 0.0)) return GSR_EINVAL;
    A->damp = damp;
    return GSR_OK;
}

int64_t gsr_debug_graph_builds(const gsr_matrix* A) { return A ? A->ws.graph_builds : 0; }

int gsr_debug_while_graph(const gsr_matrix* A) { return (A && A->ws.last_loop_while) ? 1 : 0; }

double gsr_lsqr_last_loop_ms(const gsr_matrix* A) {
    return (A && A->ws.solved) ? A->ws.last_loop_ms : -1.0;
}

int gsr_lsqr_standard_errors(gsr_matrix* A, double* se_hd, gsr_stream stream) {
    if (!A || !se_hd) return GSR_EINVAL;
    Workspace& W = A->ws;
    if (A->state != 1 || !W.solved) return GSR_ESTATE;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n = A->n_cols;
    const bool dev = is_device_ptr(se_hd);
    double* out = se_hd;
    if (!dev) {
        if (!W.stage_n) GSR_TRY(dev_alloc(A, (void**)&W.stage_n, (size_t)n * 8));
        out = W.stage_n;
    }
    const double dof = A->m_global > A->n_global ? (double)(A->m_global - A->n_global) : 1.0;
    k_standard_errors<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(W.var, A->p, W.last_rnorm, dof, out, n);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    if (!dev) {
        GSR_CUDA_TRY(cudaMemcpyAsync(se_hd, out, (size_t)n * 8, cudaMemcpyDeviceToHost, s));
        GSR_CUDA_TRY(cudaStreamSynchronize(s));
    }
    return GSR_OK;
}

int gsr_debug_fused_pass(gsr_matrix* A, const double* x_dev, double ca, double* y_dev, double* t_dev,
                         gsr_stream stream) {
    if (!A || !x_dev || !t_dev || (!y_dev && A->dims.n_rows > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    if (A->n_con > 0 || A->comm) return GSR_EUNSUPPORTED;
    cudaStream_t s = (cudaStream_t)stream;
    Workspace& W = A->ws;
    GSR_TRY(ensure_workspace(A));
    W.solved = false;
    const double coef[2] = {ca, 0.0};
    GSR_CUDA_TRY(cudaMemcpyAsync(W.red, coef, sizeof(coef), cudaMemcpyHostToDevice, s));
    GSR_CUDA_TRY(cudaStreamSynchronize(s));   // `coef` lives on this stack frame
    k_gather_sumsq<<<NB_N, TB_N, 0, s>>>(y_dev, A->perm, W.u, A->m_int, W.part_u);
    count_launch();
    GSR_TRY(launch_fused(A, x_dev, W.u, W.red, W.part_u, t_dev, nullptr, nullptr, s));
    k_sum_partials<<<1, 1024, 0, s>>>(W.part_u, A->n_units, W.red + 3, nullptr);
    GSR_TRY(launch_aprod2_instr(A, W.u, t_dev, W.red + 3, nullptr, 0, s));
    k_scatter_rows<<<NB_N, TB_N, 0, s>>>(W.u, A->perm, y_dev, A->m_int);
    count_launch(2);
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int gsr_time_product(gsr_matrix* A, int which, int reps, float* ms_avg, gsr_stream stream) {
    if (!A || !ms_avg || reps < 1 || which < 1 || which > 4) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    cudaStream_t s = (cudaStream_t)stream;
    Workspace& W = A->ws;
    GSR_TRY(ensure_workspace(A));
    cudaEvent_t e0, e1;
    GSR_CUDA_TRY(cudaEventCreate(&e0));
    GSR_CUDA_TRY(cudaEventCreate(&e1));
    int rc = GSR_OK;
    if (which == 4) {   // the instrumental pass needs a consistent u_hat and its sum of squares
        rc = launch_fused(A, W.v, W.u, A->coef_one, W.part_u, W.t, nullptr, nullptr, s);
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_u, A->n_units, W.red + 3, nullptr);
    }
    // aprod2 as the solver runs it: on one GPU with the sum of u_hat^2, which sends the instrumental
    // block through the fixed-point pass (its scale is 2^(61 - exponent of that sum)); on a row shard
    // the solver's two-pass form does not exist and the fp64 pass is what is timed.  The sum is
    // formed HERE from the u_hat in the workspace: red[3] of an earlier solve is stale once a
    // which = 1 timing has overwritten u_hat, and a wrong scale lets the conversion saturate.
    const bool with_ss = which == 2 && W.solved && !A->comm;
    if (with_ss) {
        k_sumsq<<<NB_N, TB_N, 0, s>>>(W.u, A->m_int, W.part_u, nullptr, 0, nullptr);
        k_sum_partials<<<1, 1024, 0, s>>>(W.part_u, NB_N, W.red + 3, nullptr);
    }
    for (int pass = 0; pass < 2 && rc == GSR_OK; ++pass) {   // pass 0: warm-up
        int nrep = pass == 0 ? 1 : reps;
        cudaEventRecord(e0, s);
        for (int i = 0; i < nrep && rc == GSR_OK; ++i) {
            if (which == 1) rc = launch_aprod1(A, W.v, W.u, A->coef_one, W.part_u, nullptr, nullptr, s);
            else if (which == 2)   // as the solver runs it: with the norm of u_hat of its last pass, if any
                rc = launch_aprod2(A, W.u, W.v, A->coef_one, nullptr, nullptr, s, with_ss ? W.red + 3 : nullptr);
            else if (which == 3) rc = launch_fused(A, W.v, W.u, A->coef_one, W.part_u, W.t, nullptr, nullptr, s);
            else rc = launch_aprod2_instr(A, W.u, W.t, W.red + 3, nullptr, 0, s);
        }
        cudaEventRecord(e1, s);
        if (cudaEventSynchronize(e1) != cudaSuccess) rc = GSR_ECUDA;
    }
    float ms = 0.f;
    if (rc == GSR_OK && cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) rc = GSR_ECUDA;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaGetLastError();
    *ms_avg = ms / reps;
    return rc;
}

}  // extern "C"
