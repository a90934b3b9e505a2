// aprod mode 1 and mode 2 (rows a3, a5-a8): Algorithms 1 and 2 of the paper
// on the warp-tiled, attitude-binned layout of gsr_internal.h.
//
// Kernels: k_aprod1 / k_aprod2 (the two products, also behind gsr_aprod1/2), k_fused (both in one
// read of the matrix, the solver's default iteration) and k_aprod2_instr (its instrumental pass).
// Warps are autonomous.  A persistent grid (one or two CTAs of 16 warps per SM) fetches UNITS
// (runs of 32-row tiles whose attitude blocks start inside one window of `win` knots per axis)
// from a global counter, one unit per warp at a time.  In shared memory
//     xi[0 .. I)                      the whole instrumental block, shared by the CTA's warps
//     xw[warp][0 .. 3*win)            the unit's attitude window, PRIVATE to the warp
// so the 18 irregular column accesses of a row never leave the SM; only the
// astrometric columns (5 per star, rows star-sorted inside a unit) and the global column go
// to L1/L2.  The matrix is streamed exactly once, every request coalesced.
//
// Attitude block.  Lane j < 12 of each half-warp owns COEFFICIENT j of 16 rows (the tile stores
// the 32x12 attitude block row-major, see gsr_internal.h), so for one row the 12 lanes touch
// 12 distinct, conflict-free window addresses:
//   aprod2: plain shared-memory read-modify-write, row after row, no atomics (the window is
//           private to the warp, and rows of the same warp are serialised);
//   aprod1: 12 products per row, transposed back to "lane r owns row r" by a 15-shuffle
//           butterfly inside each half-warp.
#include "gsr_internal.h"

namespace gsr {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// A tile is consumed in two phases so that the loads of one phase are in flight while the
// other phase computes (software pipeline, no extra registers):
//   phase A: the attitude block (16 coefficients per lane) + window offsets
//   phase B: astrometric, instrumental and global coefficients + star and column indices
struct RegsA {
    double at[16];             // lane (h, j): attitude coefficient min(j, 11) of rows 16h .. 16h+15
    uint32_t aoff;             // lane r: att_start - a0 of row r
};
struct RegsB {
    double as[5], in[6], gl;   // lane r: coefficients of row r
    int32_t s;
    uint32_t c[6];
};

// Streaming loads, all of a phase issued back to back (volatile asm keeps them together and
// ahead of their first use).
__device__ __forceinline__ double ld_stream_f64(const void* p) {
    double v;
    asm volatile("ld.global.cs.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ int32_t ld_stream_s32(const void* p) {
    int32_t v;
    asm volatile("ld.global.cs.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint32_t ld_stream_u16(const void* p) {
    uint16_t v;
    asm volatile("ld.global.cs.u16 %0, [%1];" : "=h"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void load_A(const unsigned char* __restrict__ T, int lane, RegsA& r) {
    r.aoff = ld_stream_u16(T + OFF_AOFF + lane * 2);
    const int h = lane >> 4, jj = min(lane & 15, 11);
#pragma unroll
    for (int q = 0; q < 16; ++q) r.at[q] = ld_stream_f64(T + OFF_ATTV + ((q * 2 + h) * 12 + jj) * 8);
}
__device__ __forceinline__ void load_B(const unsigned char* __restrict__ T, int lane, RegsB& r) {
    r.s = ld_stream_s32(T + OFF_STAR + lane * 4);
#pragma unroll
    for (int j = 0; j < 6; ++j) r.c[j] = ld_stream_u16(T + OFF_ICOL + (j * R + lane) * 2);
#pragma unroll
    for (int k = 0; k < 5; ++k) r.as[k] = ld_stream_f64(T + OFF_ASTRO + (k * R + lane) * 8);
#pragma unroll
    for (int j = 0; j < 6; ++j) r.in[j] = ld_stream_f64(T + OFF_INSTRV + (j * R + lane) * 8);
    r.gl = ld_stream_f64(T + OFF_GLOBV + lane * 8);
}

__device__ __forceinline__ void load_B_instr(const unsigned char* __restrict__ T, int lane, RegsB& r) {
#pragma unroll
    for (int j = 0; j < 6; ++j) r.c[j] = ld_stream_u16(T + OFF_ICOL + (j * R + lane) * 2);
#pragma unroll
    for (int j = 0; j < 6; ++j) r.in[j] = ld_stream_f64(T + OFF_INSTRV + (j * R + lane) * 8);
}
__device__ __forceinline__ void load_B_rest(const unsigned char* __restrict__ T, int lane, RegsB& r) {
    r.s = ld_stream_s32(T + OFF_STAR + lane * 4);
#pragma unroll
    for (int k = 0; k < 5; ++k) r.as[k] = ld_stream_f64(T + OFF_ASTRO + (k * R + lane) * 8);
    r.gl = ld_stream_f64(T + OFF_GLOBV + lane * 8);
}

__device__ __forceinline__ int fetch_unit(int* counter, int lane) {
    int u = 0;
    if (lane == 0) u = atomicAdd(counter, 1);
    return __shfl_sync(0xffffffffu, u, 0);
}

// ---- aprod1: y[i] = ca*y[i] + sum_k A[i,k] x[col(i,k)]  (Algorithm 1) --------------------
template <bool NORM, bool PERM>
__global__ void __launch_bounds__(TPB) k_aprod1(const unsigned char* __restrict__ tiles,
                                               const Unit* __restrict__ units, int n_units,
                                               int* __restrict__ counter,
                                               const double* __restrict__ x, double* __restrict__ y,
                                               const double* __restrict__ ca_p,
                                               double* __restrict__ partials,
                                               const uint32_t* __restrict__ perm, int64_t S,
                                               int64_t D, int I, int win, int ws,
                                               const int* __restrict__ stop) {
    if (stop && *stop) return;
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* xi = sm;
    double* xw = sm + ((I + 1) & ~1) + warp * 3 * ws;
    const double* xatt = x + 5 * S;
    const double* xins = x + 5 * S + 3 * D;
    for (int i = threadIdx.x; i < I; i += TPB) xi[i] = __ldg(xins + i);
    const double xg = __ldg(xins + I);
    const double ca = *ca_p;
    __syncthreads();

    const int h = lane >> 4, j = lane & 15, jj = min(j, 11);
    const int axo = (jj >> 2) * ws + (jj & 3);   // my coefficient's column, relative to aoff
    const bool att_lane = j < 12;
    for (;;) {
        const int u = fetch_unit(counter, lane);
        if (u >= n_units) break;
        const Unit un = units[u];
        __syncwarp();
        for (int i = lane; i < 3 * win; i += 32) {
            const int ax = i / win, k = i - ax * win;
            const int64_t knot = (int64_t)un.a0 + k;
            xw[ax * ws + k] = knot < D ? __ldg(xatt + ax * D + knot) : 0.0;
        }
        __syncwarp();
        double q = 0.0;
        const unsigned char* T = tiles + (int64_t)un.tile0 * TILE_BYTES;
        RegsA ra;
        load_A(T, lane, ra);
        for (int t = 0; t < un.ntiles; ++t, T += TILE_BYTES) {
            RegsB r;
            load_B(T, lane, r);
            const int64_t ri = ((int64_t)un.tile0 + t) * R + lane;
            int64_t ry = ri;
            bool live = true;
            if (PERM) {
                const uint32_t pe = __ldcs(perm + ri);
                live = pe != PERM_PAD;
                ry = pe;
            }
            const double yold = live ? __ldcs(y + ry) : 0.0;
            // phase A -- attitude: 12 lanes per row, products transposed back by a butterfly
            double p[16];
#pragma unroll
            for (int qq = 0; qq < 16; ++qq) {
                const uint32_t a = __shfl_sync(0xffffffffu, ra.aoff, h * 16 + qq);
                const double pv = ra.at[qq] * xw[a + axo];
                p[qq] = att_lane ? pv : 0.0;
            }
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) {
                const bool up = (j & o) != 0;
#pragma unroll
                for (int i = 0; i < o; ++i) {
                    const double send = up ? p[i] : p[i + o];
                    const double keep = up ? p[i + o] : p[i];
                    p[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
                }
            }
            double sum = p[0];   // lane (h, j) now holds the attitude part of row 16h + j
            if (t + 1 < un.ntiles) load_A(T + TILE_BYTES, lane, ra);   // in flight during phase B
            // phase B
            const double* xa = x + 5 * (int64_t)r.s;
#pragma unroll
            for (int k = 0; k < 5; ++k) sum = fma(r.as[k], __ldg(xa + k), sum);
#pragma unroll
            for (int k = 0; k < 6; ++k) sum = fma(r.in[k], xi[r.c[k]], sum);
            sum = fma(r.gl, xg, sum);
            const double ynew = fma(ca, yold, sum);
            if (live) y[ry] = ynew;
            if (NORM) q = fma(ynew, ynew, q);   // padding rows: y stays 0
        }
        if (NORM) {
            q = warp_sum(q);
            if (lane == 0) partials[u] = q;
        }
    }
}

// ---- aprod2: x[col(i,k)] += A[i,k] * (y[i]*sy)  (Algorithm 2) ----------------------------
// attitude block: warp-private shared-memory window, plain read-modify-write (see above),
// flushed once per unit with one global atomic per touched column; instrumental block: CTA-
// shared shared-memory accumulators (fp64 atomicAdd = CAS loop on sm_100a), flushed once per
// CTA; astrometric block: segmented warp reduction over the star-sorted rows, one global atomic
// per (warp, star, column); global column: register accumulation, one atomic per warp.
// SQUARE: accumulate A[i,k]^2 instead (column sums of squares for the preconditioner).
template <bool SQUARE, bool PERM>
__global__ void __launch_bounds__(TPB) k_aprod2(const unsigned char* __restrict__ tiles,
                                               const Unit* __restrict__ units, int n_units,
                                               int* __restrict__ counter,
                                               const double* __restrict__ y, double* __restrict__ x,
                                               const double* __restrict__ sy_p,
                                               const uint32_t* __restrict__ perm, int64_t S,
                                               int64_t D, int I, int win, int ws, int ncopy,
                                               const int* __restrict__ stop) {
    if (stop && *stop) return;
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* xi = sm;
    double* xw = sm + ((I + 1) & ~1) + warp * 3 * ws;
    double* ysm = sm + ((I + 1) & ~1) + NWARP * 3 * ws + warp * 32;   // y of the current tile: a
                                                  // shared-memory broadcast costs the LSU pipe
                                                  // less than two 32-bit shuffles per step
    // small I: one private copy of the instrumental accumulator per warp (copies 1.. behind the
    // y tiles), so that only lanes of the same instruction contend for an address (config 4)
    const int ipad = (I + 1) & ~1;
    double* xcopies = sm + ipad + NWARP * 3 * ws + NWARP * 32;
    for (int i = threadIdx.x; i < I; i += TPB) xi[i] = 0.0;
    for (int i = threadIdx.x; i < (ncopy - 1) * ipad; i += TPB) xcopies[i] = 0.0;
    if (ncopy > 1 && warp > 0) xi = xcopies + (warp - 1) * ipad;
    const double sy = SQUARE ? 1.0 : *sy_p;
    __syncthreads();

    const int h = lane >> 4, j = lane & 15, jj = min(j, 11);
    const int axo = (jj >> 2) * ws + (jj & 3);
    const bool lo12 = lane < 12, hi12 = lane >= 16 && lane < 28;
    double* xatt = x + 5 * S;
    double g = 0.0;
    for (;;) {
        const int u = fetch_unit(counter, lane);
        if (u >= n_units) break;
        const Unit un = units[u];
        __syncwarp();
        for (int i = lane; i < 3 * ws; i += 32) xw[i] = 0.0;
        __syncwarp();
        const unsigned char* T = tiles + (int64_t)un.tile0 * TILE_BYTES;
        RegsA ra;
        load_A(T, lane, ra);
        for (int t = 0; t < un.ntiles; ++t, T += TILE_BYTES) {
            RegsB r;
            load_B(T, lane, r);
            const int64_t ri = ((int64_t)un.tile0 + t) * R + lane;
            double yv = 1.0;
            if (!SQUARE) {
                if (PERM) {
                    const uint32_t pe = __ldcs(perm + ri);
                    yv = pe != PERM_PAD ? y[pe] * sy : 0.0;
                } else {
                    yv = __ldcs(y + ri) * sy;
                }
            }
            // phase A -- attitude: rows 0-15 through lanes 0-11, rows 16-31
            // through lanes 16-27, one row per half and step; the two rows of a step go in one
            // instruction unless their windows overlap (then one after the other)
            ysm[lane] = yv;
            __syncwarp();
            const uint32_t a_other = __shfl_xor_sync(0xffffffffu, ra.aoff, 16);
            const int da = (int)ra.aoff - (int)a_other;
            const unsigned cmask = __ballot_sync(0xffffffffu, da > -4 && da < 4);
#pragma unroll
            for (int qq = 0; qq < 16; ++qq) {
                const int src = h * 16 + qq;
                const uint32_t a = __shfl_sync(0xffffffffu, ra.aoff, src);
                const double yy = ysm[src];
                const double add = SQUARE ? ra.at[qq] * ra.at[qq] : ra.at[qq] * yy;
                double* pa = xw + a + axo;
                if ((cmask >> qq) & 1u) {
                    if (lo12) *pa += add;
                    __syncwarp();
                    if (hi12) *pa += add;
                } else {
                    if (lo12 || hi12) *pa += add;
                }
                __syncwarp();
            }
            if (t + 1 < un.ntiles) load_A(T + TILE_BYTES, lane, ra);   // in flight during phase B
            // phase B
#pragma unroll
            for (int k = 0; k < 5; ++k) r.as[k] = SQUARE ? r.as[k] * r.as[k] : r.as[k] * yv;
#pragma unroll
            for (int k = 0; k < 6; ++k) r.in[k] = SQUARE ? r.in[k] * r.in[k] : r.in[k] * yv;
            // instrumental
#pragma unroll
            for (int k = 0; k < 6; ++k) atomicAdd(xi + r.c[k], r.in[k]);
            // global
            g += SQUARE ? r.gl * r.gl : r.gl * yv;
            // astrometric: segmented reduction, rows are star-sorted
            const int32_t s_up = __shfl_up_sync(0xffffffffu, r.s, 1);
            const bool head = lane == 0 || s_up != r.s;
            const unsigned heads = __ballot_sync(0xffffffffu, head);
            if (heads == 1u) {   // the whole warp lies inside one star
#pragma unroll
                for (int k = 0; k < 5; ++k) {
                    const double tsum = warp_sum(r.as[k]);
                    if (lane == 0 && tsum != 0.0) atomicAdd(x + 5 * (int64_t)r.s + k, tsum);
                }
            } else {
                // segmented inclusive scan; the last lane of each segment holds its sum.  A step
                // of distance o is needed only if some run is longer than o rows, i.e. if there
                // are o consecutive non-head lanes (shuffles cost LSU data-pipe wavefronts).
                const unsigned below = heads & ((2u << lane) - 1u);        // heads at or below me
                const int seg_start = 31 - __clz(below);
                const bool tail = lane == 31 || ((heads >> (lane + 1)) & 1u);
                const unsigned n1 = ~heads, n2 = n1 & (n1 >> 1), n4 = n2 & (n2 >> 2),
                               n8 = n4 & (n4 >> 4), n16 = n8 & (n8 >> 8);
                const unsigned need = 1u | (n2 ? 2u : 0u) | (n4 ? 4u : 0u) | (n8 ? 8u : 0u) | (n16 ? 16u : 0u);
                double vs[5];
#pragma unroll
                for (int k = 0; k < 5; ++k) vs[k] = r.as[k];
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    if (need & o) {
#pragma unroll
                        for (int k = 0; k < 5; ++k) {
                            const double up = __shfl_up_sync(0xffffffffu, vs[k], o);
                            if (lane - o >= seg_start) vs[k] += up;
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < 5; ++k)
                    if (tail && vs[k] != 0.0) atomicAdd(x + 5 * (int64_t)r.s + k, vs[k]);
            }
        }
        // flush the unit's window
        __syncwarp();
        for (int i = lane; i < 3 * win; i += 32) {
            const int ax = i / win, k = i - ax * win;
            const double vacc = xw[ax * ws + k];
            if (vacc != 0.0) {
                atomicAdd(xatt + ax * D + un.a0 + k, vacc);   // knot < D whenever vacc != 0
            }
        }
    }
    // global column: one atomic per warp
    g = warp_sum(g);
    if (lane == 0 && g != 0.0) atomicAdd(x + 5 * S + 3 * D + I, g);
    // flush the CTA's instrumental accumulators
    __syncthreads();
    double* xins = x + 5 * S + 3 * D;
    for (int i = threadIdx.x; i < I; i += TPB) {
        double vacc = sm[i];
        for (int w = 1; w < ncopy; ++w) vacc += xcopies[(w - 1) * ipad + i];
        if (vacc != 0.0) atomicAdd(xins + i, vacc);
    }
}

// ---- fused LSQR pass: u <- A v + ca u  and  t += A^T u_new  in ONE read of the matrix ------
// The second half of the bidiagonalisation step needs A^T u_{k+1} = A^T u_hat / beta_{k+1}; by
// linearity the unnormalised A^T u_hat can be accumulated while u_hat is being produced, row by
// row, so the matrix is streamed once per iteration instead of twice (rows a3 + a5, a6, a8).
// The instrumental block of A^T u_hat (a7) is left to k_aprod2_instr, because its CTA-shared
// accumulator (I doubles) does not fit in shared memory beside x's instrumental block and the
// two attitude windows per warp at I = 10 000.
__global__ void __launch_bounds__(TPB) k_fused(const unsigned char* __restrict__ tiles,
                                              const Unit* __restrict__ units, int n_units,
                                              int* __restrict__ counter,
                                              const double* __restrict__ x, double* __restrict__ y,
                                              const double* __restrict__ ca_p,
                                              double* __restrict__ partials, double* __restrict__ tacc,
                                              int64_t S, int64_t D, int I, int win, int ws,
                                              const int* __restrict__ stop) {
    if (stop && *stop) return;
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* xi = sm;
    double* xw = sm + ((I + 1) & ~1) + warp * 6 * ws;   // window of v (read)
    double* tw = xw + 3 * ws;                           // window of A^T u_hat (accumulate)
    // u_hat and the window offsets of the current tile reach the attitude lanes through shared
    // memory: wide broadcast loads (two u_hat, four offsets per request) cost the LSU data pipe
    // far less than one or two 32-bit shuffles per row and step
    double* ysm = sm + ((I + 1) & ~1) + NWARP * 6 * ws + warp * 48;
    uint32_t* asm_ = (uint32_t*)(ysm + 32);
    const double* xatt = x + 5 * S;
    const double* xins = x + 5 * S + 3 * D;
    double* tatt = tacc + 5 * S;
    for (int i = threadIdx.x; i < I; i += TPB) xi[i] = __ldg(xins + i);
    const double xg = __ldg(xins + I);
    const double ca = *ca_p;
    __syncthreads();

    const int h = lane >> 4, j = lane & 15, jj = min(j, 11);
    const int axo = (jj >> 2) * ws + (jj & 3);
    const bool att_lane = j < 12;
    const bool lo12 = lane < 12, hi12 = lane >= 16 && lane < 28;
    double g = 0.0;
    for (;;) {
        const int u = fetch_unit(counter, lane);
        if (u >= n_units) break;
        const Unit un = units[u];
        __syncwarp();
        for (int i = lane; i < 3 * win; i += 32) {
            const int ax = i / win, k = i - ax * win;
            const int64_t knot = (int64_t)un.a0 + k;
            xw[ax * ws + k] = knot < D ? __ldg(xatt + ax * D + knot) : 0.0;
        }
        for (int i = lane; i < 3 * ws; i += 32) tw[i] = 0.0;
        __syncwarp();
        double q = 0.0;
        const unsigned char* T = tiles + (int64_t)un.tile0 * TILE_BYTES;
        // Loads are issued as soon as the registers they fill are dead (volatile asm keeps the
        // program order): the next tile's instrumental values and columns right after mode 1,
        // its attitude coefficients group by group inside the read-modify-write loop, the rest
        // (star, astrometric, global) at the top of its own iteration.
        RegsA ra;
        RegsB r;
        load_A(T, lane, ra);
        load_B_instr(T, lane, r);
        for (int t = 0; t < un.ntiles; ++t, T += TILE_BYTES) {
            const unsigned char* Tn = t + 1 < un.ntiles ? T + TILE_BYTES : T;   // (last: harmless reload)
            load_B_rest(T, lane, r);
            const int64_t ri = ((int64_t)un.tile0 + t) * R + lane;
            const double yold = __ldcs(y + ri);
            // ---- mode 1 for this tile
            // products of rows q and q+8 are formed together and go straight into the first
            // butterfly step, so that only 8 of the 16 partial products are ever live
            double p[8];
            asm_[lane] = ra.aoff;
            __syncwarp();
            {
                const bool up8 = (j & 8) != 0;
#pragma unroll
                for (int g4 = 0; g4 < 2; ++g4) {
                    const uint4 alo = *(const uint4*)(asm_ + h * 16 + 4 * g4);
                    const uint4 ahi = *(const uint4*)(asm_ + h * 16 + 4 * g4 + 8);
                    const uint32_t al[4] = {alo.x, alo.y, alo.z, alo.w};
                    const uint32_t ah[4] = {ahi.x, ahi.y, ahi.z, ahi.w};
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int q0 = 4 * g4 + i;
                        double plo = ra.at[q0] * xw[al[i] + axo];
                        double phi = ra.at[q0 + 8] * xw[ah[i] + axo];
                        plo = att_lane ? plo : 0.0;
                        phi = att_lane ? phi : 0.0;
                        const double send = up8 ? plo : phi;
                        const double keep = up8 ? phi : plo;
                        p[q0] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
                    }
                }
            }
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) {
                const bool up = (j & o) != 0;
#pragma unroll
                for (int i = 0; i < o; ++i) {
                    const double send = up ? p[i] : p[i + o];
                    const double keep = up ? p[i + o] : p[i];
                    p[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
                }
            }
            double sum = p[0];
            const double* xa = x + 5 * (int64_t)r.s;
#pragma unroll
            for (int k = 0; k < 5; ++k) sum = fma(r.as[k], __ldg(xa + k), sum);
#pragma unroll
            for (int k = 0; k < 6; ++k) sum = fma(r.in[k], xi[r.c[k]], sum);
            sum = fma(r.gl, xg, sum);
            const double yv = fma(ca, yold, sum);   // u_hat of this row (padding rows: 0)
            y[ri] = yv;
            ysm[lane] = yv;
            q = fma(yv, yv, q);
            load_B_instr(Tn, lane, r);
            // ---- mode 2 for this tile, attitude
            const uint32_t a_other = __shfl_xor_sync(0xffffffffu, ra.aoff, 16);
            const int da = (int)ra.aoff - (int)a_other;
            const unsigned cmask = __ballot_sync(0xffffffffu, da > -4 && da < 4);
            ra.aoff = ld_stream_u16(Tn + OFF_AOFF + lane * 2);
            __syncwarp();   // ysm visible to the whole warp
#pragma unroll
            for (int g4 = 0; g4 < 4; ++g4) {
                const uint4 a4 = *(const uint4*)(asm_ + h * 16 + 4 * g4);
                const double2 y01 = *(const double2*)(ysm + h * 16 + 4 * g4);
                const double2 y23 = *(const double2*)(ysm + h * 16 + 4 * g4 + 2);
                const uint32_t aa[4] = {a4.x, a4.y, a4.z, a4.w};
                const double yy4[4] = {y01.x, y01.y, y23.x, y23.y};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int qq = 4 * g4 + i;
                    const double add = ra.at[qq] * yy4[i];
                    double* pa = tw + aa[i] + axo;
                    if ((cmask >> qq) & 1u) {
                        if (lo12) *pa += add;
                        __syncwarp();
                        if (hi12) *pa += add;
                    } else {
                        if (lo12 || hi12) *pa += add;
                    }
                    __syncwarp();
                }
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    ra.at[4 * g4 + i] = ld_stream_f64(Tn + OFF_ATTV + (((4 * g4 + i) * 2 + h) * 12 + jj) * 8);
            }
            // ---- mode 2, global and astrometric
            g = fma(r.gl, yv, g);
#pragma unroll
            for (int k = 0; k < 5; ++k) r.as[k] *= yv;
            const int32_t s_up = __shfl_up_sync(0xffffffffu, r.s, 1);
            const bool head = lane == 0 || s_up != r.s;
            const unsigned heads = __ballot_sync(0xffffffffu, head);
            if (heads == 1u) {
#pragma unroll
                for (int k = 0; k < 5; ++k) {
                    const double tsum = warp_sum(r.as[k]);
                    if (lane == 0 && tsum != 0.0) atomicAdd(tacc + 5 * (int64_t)r.s + k, tsum);
                }
            } else {
                const unsigned below = heads & ((2u << lane) - 1u);
                const int seg_start = 31 - __clz(below);
                const bool tail = lane == 31 || ((heads >> (lane + 1)) & 1u);
                const unsigned n1 = ~heads, n2 = n1 & (n1 >> 1), n4 = n2 & (n2 >> 2),
                               n8 = n4 & (n4 >> 4), n16 = n8 & (n8 >> 8);
                const unsigned need = 1u | (n2 ? 2u : 0u) | (n4 ? 4u : 0u) | (n8 ? 8u : 0u) | (n16 ? 16u : 0u);
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    if (need & o) {
#pragma unroll
                        for (int k = 0; k < 5; ++k) {
                            const double up = __shfl_up_sync(0xffffffffu, r.as[k], o);
                            if (lane - o >= seg_start) r.as[k] += up;
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < 5; ++k)
                    if (tail && r.as[k] != 0.0) atomicAdd(tacc + 5 * (int64_t)r.s + k, r.as[k]);
            }
        }
        q = warp_sum(q);
        if (lane == 0) partials[u] = q;
        __syncwarp();
        for (int i = lane; i < 3 * win; i += 32) {
            const int ax = i / win, k = i - ax * win;
            const double vacc = tw[ax * ws + k];
            if (vacc != 0.0) atomicAdd(tatt + ax * D + un.a0 + k, vacc);
        }
    }
    g = warp_sum(g);
    if (lane == 0 && g != 0.0) atomicAdd(tacc + 5 * S + 3 * D + I, g);
}

// Instrumental block of A^T u (row a7) over the instrumental planes only (1920 B per tile):
// shared-memory accumulators, six scattered adds per row.  `ncopy` = 1: one accumulator per
// CTA; `ncopy` = NWARP (small I): one private copy per warp, so that only lanes of the same
// instruction ever contend for an address (config 4: 60 columns).
//
// FIXED = false: fp64 atomicAdd, a CAS loop on sm_100a (about 420 G adds/s on the chip).
// FIXED = true : exact 64-bit fixed-point accumulation with NATIVE 32-bit shared atomics -- low
//   word add (returns the old value, so the thread that wraps it knows), high word add with the
//   carry; integer adds commute, so the sum is exact and independent of the order (about 770 G
//   adds/s).  Only for a column-scaled matrix: every column has unit 2-norm, hence any partial
//   sum of column j is bounded by sum_i |A_ij| |y_i| <= ||A_j|| ||y|| = ||y||, and with
//   2^e >= ||y|| the scale 2^(61-e) keeps it below 2^62.  Each term is rounded once to a
//   multiple of 2^(e-61): an absolute error <= n_j 2^(e-62) per column, i.e. normwise
//   ~1e-18 ||y|| per term (fp64 atomics are componentwise accurate instead; LSQR only needs
//   the normwise bound).  ss_p points to sum y_i^2 over the rows of this launch (device).
template <bool FIXED>
__global__ void __launch_bounds__(TPB) k_aprod2_instr(const unsigned char* __restrict__ tiles,
                                                     int64_t n_tiles, const double* __restrict__ y,
                                                     double* __restrict__ xins, int I, int ncopy,
                                                     const double* __restrict__ ss_p,
                                                     const int* __restrict__ stop) {
    if (stop && *stop) return;
    extern __shared__ double sm[];
    const int ipad = (I + 1) & ~1;
    for (int i = threadIdx.x; i < ipad * ncopy; i += TPB) sm[i] = 0.0;   // +0.0 = integer 0
    int e = 0;
    if (FIXED) {
        const double ynorm = sqrt(*ss_p);
        e = ynorm > 0.0 ? ilogb(ynorm) + 1 : 0;   // 2^e > ||y||
        if (e < -900) e = -900;                   // keeps 2^(61-e) finite for a vanishing y
    }
    const double scale = FIXED ? scalbn(1.0, 61 - e) : 1.0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* acc = sm + (ncopy > 1 ? warp * ipad : 0);
    const int64_t w0 = (int64_t)blockIdx.x * NWARP + warp;
    const int64_t nw = (int64_t)gridDim.x * NWARP;
    for (int64_t tile = w0; tile < n_tiles; tile += nw) {
        const unsigned char* T = tiles + tile * TILE_BYTES;
        uint32_t c[6];
        double v[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) c[k] = ld_stream_u16(T + OFF_ICOL + (k * R + lane) * 2);
#pragma unroll
        for (int k = 0; k < 6; ++k) v[k] = ld_stream_f64(T + OFF_INSTRV + (k * R + lane) * 8);
        const double yv = __ldcs(y + tile * R + lane) * scale;
        if (FIXED) {
            unsigned* acc32 = (unsigned*)acc;
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const long long q = __double2ll_rn(v[k] * yv);
                const unsigned ql = (unsigned)q, qh = (unsigned)(q >> 32);
                const unsigned old = atomicAdd(acc32 + 2 * c[k], ql);
                const unsigned carry = (old + ql) < old ? 1u : 0u;
                if (qh + carry != 0u) atomicAdd(acc32 + 2 * c[k] + 1, qh + carry);
            }
        } else {
#pragma unroll
            for (int k = 0; k < 6; ++k) atomicAdd(acc + c[k], v[k] * yv);
        }
    }
    __syncthreads();
    const double unscale = FIXED ? scalbn(1.0, e - 61) : 1.0;
    for (int i = threadIdx.x; i < I; i += TPB) {
        double vacc;
        if (FIXED) {
            long long tot = 0;
            for (int w = 0; w < ncopy; ++w) tot += ((const long long*)sm)[w * ipad + i];
            vacc = (double)tot * unscale;
        } else {
            vacc = 0.0;
            for (int w = 0; w < ncopy; ++w) vacc += sm[w * ipad + i];
        }
        if (vacc != 0.0) atomicAdd(xins + i, vacc);
    }
}

static int instr_copies(const gsr_matrix* A) {
    return ((A->dims.n_instr + 1) / 2 * 16) * NWARP <= 96 * 1024 ? NWARP : 1;
}
static size_t instr_smem(const gsr_matrix* A) {
    return (size_t)((A->dims.n_instr + 1) / 2 * 16) * instr_copies(A);
}

template <typename K>
static int set_smem(K kernel, int bytes) {
    GSR_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    return GSR_OK;
}

template <typename K>
static int resident_ctas(K kernel, const gsr_matrix* A) {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, TPB, A->smem_bytes) != cudaSuccess) {
        cudaGetLastError();
        nb = 1;
    }
    return nb < 1 ? 1 : nb;
}

int configure_product_kernels(gsr_matrix* A) {
    const int b = A->smem_bytes;
    GSR_TRY(set_smem(k_aprod1<true, false>, b));
    GSR_TRY(set_smem(k_aprod1<false, false>, b));
    GSR_TRY(set_smem(k_aprod1<false, true>, b));
    GSR_TRY(set_smem(k_aprod2<false, false>, b));
    GSR_TRY(set_smem(k_aprod2<false, true>, b));
    GSR_TRY(set_smem(k_aprod2<true, false>, b));
    GSR_TRY(set_smem(k_fused, A->smem_fused));
    GSR_TRY(set_smem(k_aprod2_instr<false>, (int)instr_smem(A)));
    GSR_TRY(set_smem(k_aprod2_instr<true>, (int)instr_smem(A)));
    {
        int nb = 1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_fused, TPB, A->smem_fused) != cudaSuccess || nb < 1) {
            cudaGetLastError();
            nb = 1;
        }
        A->grid_fused = A->sm_count * nb;
        nb = 1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_aprod2_instr<true>, TPB, instr_smem(A)) != cudaSuccess || nb < 1) {
            cudaGetLastError();
            nb = 1;
        }
        A->grid_instr = A->sm_count * nb;
    }
    A->grid1 = A->sm_count * resident_ctas(k_aprod1<true, false>, A);
    A->grid2 = A->sm_count * resident_ctas(k_aprod2<false, false>, A);
    const int need = (A->n_units + NWARP - 1) / NWARP;
    if (A->grid1 > need) A->grid1 = need;
    if (A->grid2 > need) A->grid2 = need;
    if (A->grid_fused > need) A->grid_fused = need;
    const int64_t need_i = (A->n_tiles + NWARP - 1) / NWARP;
    if (A->grid_instr > need_i) A->grid_instr = (int)(need_i > 0 ? need_i : 1);
    return GSR_OK;
}

static int reset_counter(const gsr_matrix* A, cudaStream_t s) {
    GSR_CUDA_TRY(cudaMemsetAsync(A->unit_counter, 0, sizeof(int), s));
    return GSR_OK;
}

int launch_aprod1(const gsr_matrix* A, const double* x, double* y, const double* ca,
                  double* partials, const int* stop, const uint32_t* perm, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    const int64_t S = A->dims.n_stars, D = A->dims.n_dfa;
    const int I = (int)A->dims.n_instr;
    GSR_TRY(reset_counter(A, s));
    if (perm)
        k_aprod1<false, true><<<A->grid1, TPB, A->smem_bytes, s>>>(
            A->tiles, A->units, A->n_units, A->unit_counter, x, y, ca, nullptr, perm, S, D, I, A->win, A->wstride, stop);
    else if (partials)
        k_aprod1<true, false><<<A->grid1, TPB, A->smem_bytes, s>>>(
            A->tiles, A->units, A->n_units, A->unit_counter, x, y, ca, partials, nullptr, S, D, I, A->win, A->wstride, stop);
    else
        k_aprod1<false, false><<<A->grid1, TPB, A->smem_bytes, s>>>(
            A->tiles, A->units, A->n_units, A->unit_counter, x, y, ca, nullptr, nullptr, S, D, I, A->win, A->wstride, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_aprod2(const gsr_matrix* A, const double* y, double* x, const double* sy,
                  const int* stop, const uint32_t* perm, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    const int64_t S = A->dims.n_stars, D = A->dims.n_dfa;
    const int I = (int)A->dims.n_instr;
    GSR_TRY(reset_counter(A, s));
    if (perm)
        k_aprod2<false, true><<<A->grid2, TPB, A->smem_bytes, s>>>(
            A->tiles, A->units, A->n_units, A->unit_counter, y, x, sy, perm, S, D, I, A->win, A->wstride, instr_copies(A), stop);
    else
        k_aprod2<false, false><<<A->grid2, TPB, A->smem_bytes, s>>>(
            A->tiles, A->units, A->n_units, A->unit_counter, y, x, sy, nullptr, S, D, I, A->win, A->wstride, instr_copies(A), stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_fused(const gsr_matrix* A, const double* v, double* u, const double* ca,
                 double* partials, double* t, const int* stop, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    GSR_TRY(reset_counter(A, s));
    k_fused<<<A->grid_fused, TPB, A->smem_fused, s>>>(A->tiles, A->units, A->n_units, A->unit_counter, v, u,
                                                     ca, partials, t, A->dims.n_stars, A->dims.n_dfa,
                                                     (int)A->dims.n_instr, A->win, A->wstride, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_aprod2_instr(const gsr_matrix* A, const double* u, double* t, const double* ss,
                        const int* stop, cudaStream_t s) {
    if (A->n_tiles == 0) return GSR_OK;
    // exact fixed-point accumulation needs unit column norms (see k_aprod2_instr) and ||u||^2
    if (A->p != nullptr && ss != nullptr && !A->opt_no_fixed)
        k_aprod2_instr<true><<<A->grid_instr, TPB, instr_smem(A), s>>>(
            A->tiles, A->n_tiles, u, t + A->off_instr, (int)A->dims.n_instr, instr_copies(A), ss, stop);
    else
        k_aprod2_instr<false><<<A->grid_instr, TPB, instr_smem(A), s>>>(
            A->tiles, A->n_tiles, u, t + A->off_instr, (int)A->dims.n_instr, instr_copies(A), nullptr, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    GSR_TRY(reset_counter(A, s));
    k_aprod2<true, false><<<A->grid2, TPB, A->smem_bytes, s>>>(
        A->tiles, A->units, A->n_units, A->unit_counter, nullptr, q, nullptr, nullptr, A->dims.n_stars,
        A->dims.n_dfa, (int)A->dims.n_instr, A->win, A->wstride, instr_copies(A), nullptr);
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
    GSR_TRY(launch_aprod1(A, x_dev, y_dev, A->coef_one, nullptr, nullptr, A->perm, (cudaStream_t)stream));
    return launch_con_aprod1(A, x_dev, y_dev + A->dims.n_rows, A->coef_one, nullptr, nullptr, (cudaStream_t)stream);
}

int gsr_aprod2(const gsr_matrix* A, const double* y_dev, double* x_dev, gsr_stream stream) {
    if (!A || !x_dev || (!y_dev && A->dims.n_rows > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    GSR_TRY(launch_aprod2(A, y_dev, x_dev, A->coef_one, nullptr, A->perm, (cudaStream_t)stream));
    return launch_con_aprod2(A, y_dev + A->dims.n_rows, x_dev, A->coef_one, nullptr, (cudaStream_t)stream);
}

}  // extern "C"
