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
// to L1/L2.  The matrix is streamed exactly once, every request covers whole 128-byte lines.
//
// Attitude block.  Lane (h, j), j < 12, of each half-warp owns COEFFICIENT j of the 16 attitude
// slots of its half (gsr_internal.h), so for one slot the 12 lanes touch 12 distinct,
// conflict-free window addresses:
//   aprod2: plain shared-memory read-modify-write, slot after slot, no atomics (the window is
//           private to the warp, and slots of the same warp are serialised);
//   aprod1: 12 products per slot, summed over the 12 lanes by fp64 tensor-core MMAs with
//           constant 0/1 operands (reduce_slots) -- no shuffles, nothing on the LSU pipe.
#include "gsr_internal.h"

// compute-sanitizer is closed on the GPU pool this was developed on: -DGSR_BOUNDS_CHECK turns the
// index computations of the product kernels into device asserts instead.
#ifdef GSR_BOUNDS_CHECK
#include <assert.h>
#define GSR_ASSERT(c) assert(c)
#else
#define GSR_ASSERT(c) ((void)0)
#endif

// Cache qualifier of the loads that stream the tiles (-DGSR_LDQ=... to measure another one).
// Measured on B200 at cfg2/cfg3: ".cs" (evict-first) = ".L1::no_allocate" = ".nc.L1::no_allocate"
// = ".cv" within 1 %, ".lu" 2 % slower.
#ifndef GSR_LDQ
#define GSR_LDQ ".cs"
#endif

namespace gsr {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// D(8x8) += A(8x4) B(4x8), fp64 (DMMA).  Fragments: lane l holds A[l>>2][l&3], B[l&3][l>>2] and
// D[l>>2][2(l&3) + {0,1}].
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// Lane (h, j) = 16h + j holds p[q], its term of attitude slot (h, q), q < 16 (lanes j >= 12
// hold zeros).  Returns, in lane l, the sum over the 12 lanes of the slot att_slot(l).
//   stage 1, one MMA per q:  D1_b[q&7][n] += sum_k [p of lane 4n+k][q]   (A = row selector,
//            B = the terms; n = lane group = (h, axis), k = knot: the sum over the 4 knots)
//   stage 2, four MMAs:      S[i][q'] = sum over the 4 lane groups of half (i&1) of D1_b[q'][.]
//            with b = (i>>1)&1; rows i and i+4 are duplicates, so that every lane finds one slot
//            sum in its own D fragment: of the lanes l, l ^ 16 one takes column 2(l&3), the other the
//            next (att_slot() in gsr_internal.h says which).
// Four independent accumulator chains in stage 1 and two in stage 2 keep the dependent depth at
// 4 + 2 MMAs.  The MMAs run on the fp64 tensor pipe (4 cycles each per SM, measured), which is
// otherwise idle; the 15-shuffle butterfly this replaces cost 30 LSU wavefronts per tile.
__device__ __forceinline__ double reduce_slots(const double (&p)[16], int lane) {
    const int grp = lane >> 2;
    double d1[4][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};   // [b + 2 * (q & 1)]
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const double sel = __hiloint2double(grp == (q & 7) ? 0x3FF00000 : 0, 0);
        const int c = (q >> 3) + 2 * (q & 1);
        dmma(d1[c][0], d1[c][1], sel, p[q]);
    }
    double s[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
    for (int b = 0; b < 2; ++b) {
        const double a2 = __hiloint2double((grp & 3) == 2 * b + ((lane & 3) >> 1) ? 0x3FF00000 : 0, 0);
        dmma(s[b][0], s[b][1], a2, d1[b][0] + d1[b + 2][0]);
        dmma(s[b][0], s[b][1], a2, d1[b][1] + d1[b + 2][1]);
    }
    return ((lane >> 4) ^ ((lane >> 2) & 1)) ? s[0][1] + s[1][1] : s[0][0] + s[1][0];   // see att_slot()
}

// A tile is consumed in two phases so that the loads of one phase are in flight while the
// other phase computes (software pipeline, no extra registers):
//   phase A: the attitude block (16 coefficients per lane) + window offsets
//   phase B: astrometric, instrumental and global coefficients + star and column indices
struct RegsA {
    double at[16];             // lane (h, j): attitude coefficient j of slots (h, 0 .. 15); j >= 12: 0
    uint32_t aw[4];            // the 16 window offsets (u8) of the slots of half h
    uint32_t cmask;            // bit q: slots (0, q) and (1, q) overlap
};
struct RegsB {
    double as[5], in[6], gl;   // home lane l: coefficients of row l
    int32_t s;
    uint32_t cw[3];            // instrumental columns, two per word
};
__device__ __forceinline__ uint32_t aoff_of(const uint32_t (&aw)[4], int q) {
    return (aw[q >> 2] >> (8 * (q & 3))) & 0xffu;
}
__device__ __forceinline__ uint32_t icol_of(const uint32_t (&cw)[3], int j) {
    return (j & 1) ? cw[j >> 1] >> 16 : cw[j >> 1] & 0xffffu;
}

// Streaming loads, all of a phase issued back to back (volatile asm keeps them together and
// ahead of their first use).
__device__ __forceinline__ double ld_stream_f64(const void* p) {
    double v;
    asm volatile("ld.global" GSR_LDQ ".f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ int32_t ld_stream_s32(const void* p) {
    int32_t v;
    asm volatile("ld.global" GSR_LDQ ".s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint32_t ld_stream_u32(const void* p) {
    uint32_t v;
    asm volatile("ld.global" GSR_LDQ ".u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
// two attitude coefficients (slots 2i, 2i+1); lanes j >= 12 keep their zeros
__device__ __forceinline__ void ld_att_pair(const void* p, int active, double& a, double& b) {
    asm volatile("{\n\t.reg .pred pa;\n\tsetp.ne.s32 pa, %2, 0;\n\t"
                 "@pa ld.global" GSR_LDQ ".v2.f64 {%0, %1}, [%3];\n\t}"
                 : "+d"(a), "+d"(b) : "r"(active), "l"(p));
}
__device__ __forceinline__ void ld_aoff(const unsigned char* T, int h, uint32_t (&aw)[4]) {
    asm volatile("ld.global" GSR_LDQ ".v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(aw[0]), "=r"(aw[1]), "=r"(aw[2]), "=r"(aw[3]) : "l"(T + OFF_AOFF + h * 16));
}
__device__ __forceinline__ void load_A(const unsigned char* __restrict__ T, int lane, RegsA& r) {
    const int h = lane >> 4, jj = min(lane & 15, 11), act = (lane & 15) < 12;
    ld_aoff(T, h, r.aw);
    r.cmask = ld_stream_u32(T + OFF_CMASK);
#pragma unroll
    for (int i = 0; i < 8; ++i)
        ld_att_pair(T + OFF_ATTV + ((i * 2 + h) * 12 + jj) * 16, act, r.at[2 * i], r.at[2 * i + 1]);
}
__device__ __forceinline__ void zero_A(RegsA& r) {
#pragma unroll
    for (int q = 0; q < 16; ++q) r.at[q] = 0.0;
}
__device__ __forceinline__ void load_B_instr(const unsigned char* __restrict__ T, int lane, RegsB& r) {
#pragma unroll
    for (int j = 0; j < 3; ++j) r.cw[j] = ld_stream_u32(T + OFF_ICOL + (j * R + lane) * 4);
#pragma unroll
    for (int j = 0; j < 6; ++j) r.in[j] = ld_stream_f64(T + OFF_INSTRV + (j * R + lane) * 8);
}
__device__ __forceinline__ void load_B_rest(const unsigned char* __restrict__ T, int lane, RegsB& r) {
    r.s = ld_stream_s32(T + OFF_STAR + lane * 4);
#pragma unroll
    for (int k = 0; k < 5; ++k) r.as[k] = ld_stream_f64(T + OFF_ASTRO + (k * R + lane) * 8);
    r.gl = ld_stream_f64(T + OFF_GLOBV + lane * 8);
}
__device__ __forceinline__ void load_B(const unsigned char* __restrict__ T, int lane, RegsB& r) {
    load_B_rest(T, lane, r);
    load_B_instr(T, lane, r);
}

// fp64 add to shared memory.  sm_100a has no native fp64 (or 64-bit add) shared atomic; the
// builtin atomicAdd(double*) is expanded by ptxas into an LDS + ATOMS.CAST.SPIN loop AFTER its
// convergence analysis, and with this file's kernels it came out without the reconvergence
// barrier around the loop (lanes that lost a round were still spinning when the rest of the
// warp went on to the segmented-scan shuffles).  An explicit compare-and-swap loop keeps the
// divergence visible to the compiler.
__device__ __forceinline__ void smem_add_f64(double* addr, double v) {
    unsigned long long* a = (unsigned long long*)addr;
    unsigned long long old = *a, assumed;
    do {
        assumed = old;
        old = atomicCAS(a, assumed, (unsigned long long)__double_as_longlong(v + __longlong_as_double((long long)assumed)));
    } while (assumed != old);
}

// Bulk L2 prefetch (TMA unit, one instruction from one lane, nothing on the LSU pipe): the
// tile PF_TILES ahead and its slice of the m-sized vector are on their way to L2 while the warp
// works, so that the register loads issued one tile ahead find their lines there (about 300
// cycles away instead of HBM's 800+).  Bytes in flight no longer depend on registers.
constexpr int PF_TILES = 2;
__device__ __forceinline__ void prefetch_l2(const void* p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

__device__ __forceinline__ int fetch_unit(int* counter, int lane) {
    int u = 0;
    if (lane == 0) u = atomicAdd(counter, 1);
    return __shfl_sync(0xffffffffu, u, 0);
}

// attitude part of aprod1 for one tile: lane l returns the attitude sum of its own row
__device__ __forceinline__ double att_mode1(const RegsA& ra, const double* xw, int axo, int lane) {
    double p[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) p[q] = ra.at[q] * xw[aoff_of(ra.aw, q) + axo];
    return reduce_slots(p, lane);
}

// attitude part of aprod2 for one slot pair: slot (0, q) through lanes 0-11,
// slot (1, q) through lanes 16-27, one slot per half and step; the two slots of a step go in
// one instruction unless their windows overlap (cmask; then one after the other).  CHECK =
// false: the tile has no overlapping pair (cmask == 0, about half of all tiles), no test per
// step.  SQUARE: add the squared coefficients instead.
template <bool SQUARE, bool CHECK>
__device__ __forceinline__ void att_mode2_step(const RegsA& ra, int q, double yy, double* tw, int axo,
                                               bool lo12, bool hi12, int ws_dbg) {
    double* pa = tw + aoff_of(ra.aw, q) + axo;
    GSR_ASSERT((int)aoff_of(ra.aw, q) + 3 < ws_dbg);
    const double c = ra.at[q];
    if (CHECK && ((ra.cmask >> q) & 1u)) {
        if (lo12) *pa = SQUARE ? fma(c, c, *pa) : fma(c, yy, *pa);
        __syncwarp();
        if (hi12) *pa = SQUARE ? fma(c, c, *pa) : fma(c, yy, *pa);
    } else {
        if (lo12 || hi12) *pa = SQUARE ? fma(c, c, *pa) : fma(c, yy, *pa);
    }
    __syncwarp();
}

// the 16 steps of one tile; NEXT: reload the attitude coefficients of the next tile (Tn) pair by
// pair as soon as their registers are dead (k_fused)
template <bool SQUARE, bool CHECK, bool NEXT>
__device__ __forceinline__ void att_mode2_tile(RegsA& ra, const double* ysm, double* tw, int axo, int lane,
                                               const unsigned char* Tn, int ws_dbg) {
    const int h = lane >> 4, jj = min(lane & 15, 11), act = (lane & 15) < 12;
    const bool lo12 = lane < 12, hi12 = lane >= 16 && lane < 28;
#pragma unroll
    for (int g4 = 0; g4 < 4; ++g4) {
        double yy4[4] = {0.0, 0.0, 0.0, 0.0};
        if (!SQUARE) {
            const double2 y01 = *(const double2*)(ysm + h * 16 + 4 * g4);
            const double2 y23 = *(const double2*)(ysm + h * 16 + 4 * g4 + 2);
            yy4[0] = y01.x; yy4[1] = y01.y; yy4[2] = y23.x; yy4[3] = y23.y;
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
            att_mode2_step<SQUARE, CHECK>(ra, 4 * g4 + i, yy4[i], tw, axo, lo12, hi12, ws_dbg);
        if (NEXT) {
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int ip = 2 * g4 + i;
                ld_att_pair(Tn + OFF_ATTV + ((ip * 2 + h) * 12 + jj) * 16, act, ra.at[2 * ip], ra.at[2 * ip + 1]);
            }
        }
    }
}

// GSR_OPT_DETERMINISTIC: every sum that leaves a warp goes to global memory as a 64-bit fixed-
// point integer (native L2 integer atomics: integer addition is associative, so the result does
// not depend on the order in which warps arrive).  On a column-scaled matrix every partial sum
// of column j is bounded by sum_i |A_ij| |u_i| <= ||A_j|| ||u|| = ||u||; with 2^e >= ||u|| the
// scale 2^(61-e) keeps it below 2^62.  What a warp adds is itself deterministic: a unit's rows
// are processed in a fixed order by one warp.
template <bool DET>
__device__ __forceinline__ void add_out(double* addr, double v, double dscale) {
    if (DET) atomicAdd((unsigned long long*)addr, (unsigned long long)__double2ll_rn(v * dscale));
    else atomicAdd(addr, v);
}
// exponent e with 2^e > sqrt(ss) (the norm of the vector whose A^T product is accumulated)
__device__ __forceinline__ int fixed_exp(double ss) {
    const double ynorm = sqrt(ss);
    int e = ynorm > 0.0 ? ilogb(ynorm) + 1 : 0;
    return e < -900 ? -900 : e;   // keeps 2^(61-e) finite for a vanishing vector
}

// astrometric part of aprod2 for one tile: segmented reduction over the
// star-sorted home lanes, one global atomic per (tile, star, coefficient).  vs[k] = A[l,k]*y[l].
// (Measured on B200, cfg3, real LSQR vectors: cutting the runs into pieces of 8 / 4 / 2 / 1 rows to
// save scan steps -- 1 = one atomic per row and coefficient, no scan -- gives k_fused 13.9 / 13.9 /
// 14.8 / 18.3 ms against 13.9 for whole runs: the L2 atomic rate, not the shuffles, is what the
// shorter pieces run into.  Timed with u = 0 the same variants look 6 % FASTER, because the
// zero-valued atomics are skipped: product timings need real vectors.)
template <bool DET>
__device__ __forceinline__ void astro_mode2(double (&vs)[5], int32_t s, int lane, double* __restrict__ x,
                                            int64_t S, double dscale) {
    GSR_ASSERT(s >= 0 && s < S);
    const int32_t s_up = __shfl_up_sync(0xffffffffu, s, 1);
    const bool head = lane == 0 || s_up != s;
    const unsigned heads = __ballot_sync(0xffffffffu, head);
    if (heads == 1u) {   // the whole warp lies inside one star
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const double tsum = warp_sum(vs[k]);
            if (lane == 0 && tsum != 0.0) add_out<DET>(x + 5 * (int64_t)s + k, tsum, dscale);
        }
    } else {
        // segmented inclusive scan; the last lane of each segment holds its sum.  A step of
        // distance o is needed only if some run is longer than o rows, i.e. if there are o
        // consecutive non-head lanes (shuffles cost LSU data-pipe wavefronts).
        const unsigned below = heads & ((2u << lane) - 1u);        // heads at or below me
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
                    const double up = __shfl_up_sync(0xffffffffu, vs[k], o);
                    if (lane - o >= seg_start) vs[k] += up;
                }
            }
        }
#pragma unroll
        for (int k = 0; k < 5; ++k)
            if (tail && vs[k] != 0.0) add_out<DET>(x + 5 * (int64_t)s + k, vs[k], dscale);
    }
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

    const int jj = min(lane & 15, 11);
    const int axo = (jj >> 2) * ws + (jj & 3);   // my coefficient's column, relative to aoff
    RegsA ra;
    zero_A(ra);
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
        load_A(T, lane, ra);
        if (lane == 0 && un.ntiles > 1) prefetch_l2(T + TILE_BYTES, TILE_BYTES);
        for (int t = 0; t < un.ntiles; ++t, T += TILE_BYTES) {
            RegsB r;
            load_B(T, lane, r);
            const int64_t ri = ((int64_t)un.tile0 + t) * R + lane;
            if (lane == 0 && t + PF_TILES < un.ntiles) {
                prefetch_l2(T + PF_TILES * TILE_BYTES, TILE_BYTES);
                if (!PERM) prefetch_l2(y + ri + PF_TILES * R, R * 8);
            }
            int64_t ry = ri;
            bool live = true;
            if (PERM) {
                const uint32_t pe = __ldcs(perm + ri);
                live = pe != PERM_PAD;
                ry = pe;
            }
            const double yold = live ? __ldcs(y + ry) : 0.0;
            // phase A -- attitude
            double sum = att_mode1(ra, xw, axo, lane);
            if (t + 1 < un.ntiles) load_A(T + TILE_BYTES, lane, ra);   // in flight during phase B
            // phase B
            const double* xa = x + 5 * (int64_t)r.s;
#pragma unroll
            for (int k = 0; k < 5; ++k) sum = fma(r.as[k], __ldg(xa + k), sum);
#pragma unroll
            for (int k = 0; k < 6; ++k) sum = fma(r.in[k], xi[icol_of(r.cw, k)], sum);
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
// INSTR = false: the instrumental block is left to k_aprod2_instr, which reads only the 1920
// instrumental bytes of every tile (the split the fused iteration uses, section 5.4 of DESIGN.md):
// the six compare-and-swap adds per row no longer share the LSU data pipe with the attitude
// read-modify-writes, and this kernel streams 152 instead of 212 bytes per row.  With PERM the
// scaled y of every internal row is also written to yint, so that the instrumental pass reads it
// contiguously instead of gathering it a second time.
// Warps per CTA of the main launch (INSTR = false).  Without the instrumental accumulators that
// launch is bound by the latency of its serial per-tile chains, not by a pipe (ncu at 16 warps:
// LSU 68 %, DRAM 65 %), and with 24 warps it still fits the register file (80 registers, no
// spills) and shared memory (24 windows).  Measured at cfg3, main launch + fixed-point pass:
// 13.9 / 13.1 / 12.7 / 13.4 ms for 16 / 20 / 24 / 28 warps.
#ifndef GSR_NW_MAIN
#define GSR_NW_MAIN 24
#endif
constexpr int NWARP_MAIN = GSR_NW_MAIN;
template <bool SQUARE, bool PERM, bool INSTR>
__global__ void __launch_bounds__(INSTR ? TPB : NWARP_MAIN * 32) k_aprod2(const unsigned char* __restrict__ tiles,
                                               const Unit* __restrict__ units, int n_units,
                                               int* __restrict__ counter,
                                               const double* __restrict__ y, double* __restrict__ x,
                                               const double* __restrict__ sy_p,
                                               const uint32_t* __restrict__ perm, int64_t S,
                                               int64_t D, int I, int win, int ws, int ncopy,
                                               const int* __restrict__ stop, double* __restrict__ yint) {
    if (stop && *stop) return;
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ipad = INSTR ? (I + 1) & ~1 : 0;
    constexpr int NW = INSTR ? NWARP : NWARP_MAIN;
    double* xi = sm;
    double* xw = sm + ipad + warp * 3 * ws;
    double* ysm = sm + ipad + NW * 3 * ws + warp * 32;   // y of the current tile by
                                                  // attitude slot: wide shared-memory broadcasts
                                                  // cost the LSU pipe less than shuffles
    // small I: one private copy of the instrumental accumulator per warp (copies 1.. behind the
    // y tiles), so that only lanes of the same instruction contend for an address (config 4)
    double* xcopies = sm + ipad + NW * 3 * ws + NW * 32;
    if (INSTR) {
        for (int i = threadIdx.x; i < I; i += TPB) xi[i] = 0.0;
        for (int i = threadIdx.x; i < (ncopy - 1) * ipad; i += TPB) xcopies[i] = 0.0;
        if (ncopy > 1 && warp > 0) xi = xcopies + (warp - 1) * ipad;
    }
    const double sy = SQUARE ? 1.0 : *sy_p;
    __syncthreads();

    const int jj = min(lane & 15, 11);
    const int axo = (jj >> 2) * ws + (jj & 3);
    const int myslot = att_slot(lane);
    double* xatt = x + 5 * S;
    double g = 0.0;
    RegsA ra;
    zero_A(ra);
    for (;;) {
        const int u = fetch_unit(counter, lane);
        if (u >= n_units) break;
        const Unit un = units[u];
        __syncwarp();
        for (int i = lane; i < 3 * ws; i += 32) xw[i] = 0.0;
        __syncwarp();
        const unsigned char* T = tiles + (int64_t)un.tile0 * TILE_BYTES;
        load_A(T, lane, ra);
        if (lane == 0 && un.ntiles > 1) prefetch_l2(T + TILE_BYTES, TILE_BYTES);
        for (int t = 0; t < un.ntiles; ++t, T += TILE_BYTES) {
            RegsB r;
            if (INSTR) load_B(T, lane, r);
            else load_B_rest(T, lane, r);
            const int64_t ri = ((int64_t)un.tile0 + t) * R + lane;
            if (lane == 0 && t + PF_TILES < un.ntiles) {
                // (!INSTR: the two halves of the record this kernel reads, not the instrumental part)
                if (INSTR) {
                    prefetch_l2(T + PF_TILES * TILE_BYTES, TILE_BYTES);
                } else {
                    prefetch_l2(T + PF_TILES * TILE_BYTES, OFF_INSTRV);
                    prefetch_l2(T + PF_TILES * TILE_BYTES + OFF_GLOBV, TILE_BYTES - OFF_GLOBV);
                }
                if (!SQUARE && !PERM) prefetch_l2(y + ri + PF_TILES * R, R * 8);
            }
            double yv = 1.0;
            if (!SQUARE) {
                if (PERM) {
                    const uint32_t pe = __ldcs(perm + ri);
                    yv = pe != PERM_PAD ? y[pe] * sy : 0.0;
                    if (!INSTR) yint[ri] = yv;
                } else {
                    yv = __ldcs(y + ri) * sy;
                }
                ysm[myslot] = yv;
                __syncwarp();
            }
            // phase A -- attitude
            if (ra.cmask == 0u) att_mode2_tile<SQUARE, false, false>(ra, ysm, xw, axo, lane, nullptr, win);
            else att_mode2_tile<SQUARE, true, false>(ra, ysm, xw, axo, lane, nullptr, win);
            if (t + 1 < un.ntiles) load_A(T + TILE_BYTES, lane, ra);   // in flight during phase B
            // phase B
#pragma unroll
            for (int k = 0; k < 5; ++k) r.as[k] = SQUARE ? r.as[k] * r.as[k] : r.as[k] * yv;
            // instrumental
            if (INSTR) {
#pragma unroll
                for (int k = 0; k < 6; ++k) r.in[k] = SQUARE ? r.in[k] * r.in[k] : r.in[k] * yv;
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    GSR_ASSERT((int)icol_of(r.cw, k) < I);
                    smem_add_f64(xi + icol_of(r.cw, k), r.in[k]);
                }
                __syncwarp();
            }
            // global
            g += SQUARE ? r.gl * r.gl : r.gl * yv;
            astro_mode2<false>(r.as, r.s, lane, x, S, 1.0);
        }
        // flush the unit's window
        __syncwarp();
        for (int i = lane; i < 3 * win; i += 32) {
            const int ax = i / win, k = i - ax * win;
            const double vacc = xw[ax * ws + k];
            if (vacc != 0.0 && un.a0 + k < D) atomicAdd(xatt + ax * D + un.a0 + k, vacc);
        }
    }
    // global column: one atomic per warp
    g = warp_sum(g);
    if (lane == 0 && g != 0.0) atomicAdd(x + 5 * S + 3 * D + I, g);
    // flush the CTA's instrumental accumulators
    if (INSTR) {
        __syncthreads();
        double* xins = x + 5 * S + 3 * D;
        for (int i = threadIdx.x; i < I; i += TPB) {
            double vacc = sm[i];
            for (int w = 1; w < ncopy; ++w) vacc += xcopies[(w - 1) * ipad + i];
            if (vacc != 0.0) atomicAdd(xins + i, vacc);
        }
    }
}

// ---- fused LSQR pass: u <- A v + ca u  and  t += A^T u_new  in ONE read of the matrix ------
// The second half of the bidiagonalisation step needs A^T u_{k+1} = A^T u_hat / beta_{k+1}; by
// linearity the unnormalised A^T u_hat can be accumulated while u_hat is being produced, row by
// row, so the matrix is streamed once per iteration instead of twice (rows a3 + a5, a6, a8).
// The instrumental block of A^T u_hat (a7) is left to k_aprod2_instr, because its CTA-shared
// accumulator (I doubles) does not fit in shared memory beside x's instrumental block and the
// two attitude windows per warp at I = 10 000.
// DET (GSR_OPT_DETERMINISTIC): t is accumulated as 64-bit fixed-point integers with the scale
// 2^(61 - *det_e) (see add_out), the global column once per unit instead of once per warp.
template <bool DET>
__global__ void __launch_bounds__(TPB) k_fused(const unsigned char* __restrict__ tiles,
                                              const Unit* __restrict__ units, int n_units,
                                              int* __restrict__ counter,
                                              const double* __restrict__ x, double* __restrict__ y,
                                              const double* __restrict__ ca_p,
                                              double* __restrict__ partials, double* __restrict__ tacc,
                                              int64_t S, int64_t D, int I, int win, int ws,
                                              const int* __restrict__ stop, const int* __restrict__ det_e) {
    if (stop && *stop) return;
    const double dscale = DET ? scalbn(1.0, 61 - *det_e) : 1.0;
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* xi = sm;
    double* xw = sm + ((I + 1) & ~1) + warp * 6 * ws;   // window of v (read)
    double* tw = xw + 3 * ws;                           // window of A^T u_hat (accumulate)
    // u_hat of the current tile reaches the attitude lanes through shared memory (by attitude
    // slot): wide broadcast loads, two u_hat per request, cost the LSU data pipe far less than
    // two 32-bit shuffles per slot
    double* ysm = sm + ((I + 1) & ~1) + NWARP * 6 * ws + warp * 48;
    const double* xatt = x + 5 * S;
    const double* xins = x + 5 * S + 3 * D;
    double* tatt = tacc + 5 * S;
    for (int i = threadIdx.x; i < I; i += TPB) xi[i] = __ldg(xins + i);
    const double xg = __ldg(xins + I);
    const double ca = *ca_p;
    __syncthreads();

    const int h = lane >> 4, jj = min(lane & 15, 11);
    const int axo = (jj >> 2) * ws + (jj & 3);
    const int myslot = att_slot(lane);
    double g = 0.0;
    RegsA ra;
    zero_A(ra);
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
        // program order): the next tile's window offsets, instrumental values and columns right
        // after mode 1, its attitude coefficients pair by pair inside the read-modify-write
        // loop, the rest (star, astrometric, global) at the top of its own iteration.
        RegsB r;
        load_A(T, lane, ra);
        load_B_instr(T, lane, r);
        if (lane == 0 && un.ntiles > 1) prefetch_l2(T + TILE_BYTES, TILE_BYTES);
        for (int t = 0; t < un.ntiles; ++t, T += TILE_BYTES) {
            const unsigned char* Tn = t + 1 < un.ntiles ? T + TILE_BYTES : T;   // (last: harmless reload)
            load_B_rest(T, lane, r);
            const int64_t ri = ((int64_t)un.tile0 + t) * R + lane;
            if (lane == 0 && t + PF_TILES < un.ntiles) {
                prefetch_l2(T + PF_TILES * TILE_BYTES, TILE_BYTES);
                prefetch_l2(y + ri + PF_TILES * R, R * 8);
            }
            const double yold = __ldcs(y + ri);
            // ---- mode 1 for this tile
            double sum = att_mode1(ra, xw, axo, lane);
            uint32_t awn[4];
            ld_aoff(Tn, h, awn);
            const uint32_t cmaskn = ld_stream_u32(Tn + OFF_CMASK);
            const double* xa = x + 5 * (int64_t)r.s;
#pragma unroll
            for (int k = 0; k < 5; ++k) sum = fma(r.as[k], __ldg(xa + k), sum);
#pragma unroll
            for (int k = 0; k < 6; ++k) sum = fma(r.in[k], xi[icol_of(r.cw, k)], sum);
            sum = fma(r.gl, xg, sum);
            const double yv = fma(ca, yold, sum);   // u_hat of this row (padding rows: 0)
            y[ri] = yv;
            ysm[myslot] = yv;
            q = fma(yv, yv, q);
            load_B_instr(Tn, lane, r);
            __syncwarp();   // ysm visible to the whole warp
            // ---- mode 2 for this tile, attitude
            if (ra.cmask == 0u) att_mode2_tile<false, false, true>(ra, ysm, tw, axo, lane, Tn, win);
            else att_mode2_tile<false, true, true>(ra, ysm, tw, axo, lane, Tn, win);
#pragma unroll
            for (int i = 0; i < 4; ++i) ra.aw[i] = awn[i];
            ra.cmask = cmaskn;
            // ---- mode 2, global and astrometric
            g = fma(r.gl, yv, g);
#pragma unroll
            for (int k = 0; k < 5; ++k) r.as[k] *= yv;
            astro_mode2<DET>(r.as, r.s, lane, tacc, S, dscale);
        }
        q = warp_sum(q);
        if (lane == 0) partials[u] = q;
        __syncwarp();
        for (int i = lane; i < 3 * win; i += 32) {
            const int ax = i / win, k = i - ax * win;
            const double vacc = tw[ax * ws + k];
            if (vacc != 0.0 && un.a0 + k < D) add_out<DET>(tatt + ax * D + un.a0 + k, vacc, dscale);
        }
        if (DET) {   // the unit -> warp assignment is dynamic: one sum per unit, not per warp
            g = warp_sum(g);
            if (lane == 0 && g != 0.0) add_out<true>(tacc + 5 * S + 3 * D + I, g, dscale);
            g = 0.0;
        }
    }
    if (!DET) {
        g = warp_sum(g);
        if (lane == 0 && g != 0.0) atomicAdd(tacc + 5 * S + 3 * D + I, g);
    }
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
// det (FIXED only): leave the integer totals in xins (64-bit integer atomics, scale 2^(61-e)
// with e = fixed_exp(*ss_p)); k_det_finish converts the vector afterwards.
template <bool FIXED>
__global__ void __launch_bounds__(TPB) k_aprod2_instr(const unsigned char* __restrict__ tiles,
                                                     int64_t n_tiles, const double* __restrict__ y,
                                                     double* __restrict__ xins, int I, int ncopy,
                                                     const double* __restrict__ ss_p,
                                                     const int* __restrict__ stop, int det,
                                                     const double* __restrict__ sy_p) {
    if (stop && *stop) return;
    extern __shared__ double sm[];
    const int ipad = (I + 1) & ~1;
    for (int i = threadIdx.x; i < ipad * ncopy; i += TPB) sm[i] = 0.0;   // +0.0 = integer 0
    const int e = FIXED ? fixed_exp(*ss_p) : 0;   // 2^e > ||y||
    // sy_p (the stand-alone product only): the product is A^T (y * *sy_p); FIXED applies the factor
    // to the totals, so that the range bound stays ||y||
    const double scale = FIXED ? scalbn(1.0, 61 - e) : (sy_p ? *sy_p : 1.0);
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* acc = sm + (ncopy > 1 ? warp * ipad : 0);
    const int64_t w0 = (int64_t)blockIdx.x * NWARP + warp;
    const int64_t nw = (int64_t)gridDim.x * NWARP;
    for (int64_t tile = w0; tile < n_tiles; tile += nw) {
        const unsigned char* T = tiles + tile * TILE_BYTES;
        uint32_t cw[3], c[6];
        double v[6];
#pragma unroll
        for (int k = 0; k < 3; ++k) cw[k] = ld_stream_u32(T + OFF_ICOL + (k * R + lane) * 4);
#pragma unroll
        for (int k = 0; k < 6; ++k) v[k] = ld_stream_f64(T + OFF_INSTRV + (k * R + lane) * 8);
#pragma unroll
        for (int k = 0; k < 6; ++k) c[k] = icol_of(cw, k);
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
            for (int k = 0; k < 6; ++k) smem_add_f64(acc + c[k], v[k] * yv);
            __syncwarp();
        }
    }
    __syncthreads();
    const double unscale = FIXED ? scalbn(1.0, e - 61) * (sy_p ? *sy_p : 1.0) : 1.0;
    for (int i = threadIdx.x; i < I; i += TPB) {
        double vacc;
        if (FIXED) {
            long long tot = 0;
            for (int w = 0; w < ncopy; ++w) tot += ((const long long*)sm)[w * ipad + i];
            if (det) {
                if (tot != 0) atomicAdd((unsigned long long*)(xins + i), (unsigned long long)tot);
                continue;
            }
            vacc = (double)tot * unscale;
        } else {
            vacc = 0.0;
            for (int w = 0; w < ncopy; ++w) vacc += sm[w * ipad + i];
        }
        if (vacc != 0.0) atomicAdd(xins + i, vacc);
    }
}

// GSR_OPT_DETERMINISTIC: t holds 64-bit fixed-point integers after k_fused<true> (scale
// 2^(61 - *det_e)) and the deterministic instrumental pass (scale from *ss_p); back to doubles.
__global__ void __launch_bounds__(256) k_det_finish(double* __restrict__ t, int64_t n, int64_t off_instr,
                                                    int64_t I, const int* __restrict__ det_e,
                                                    const double* __restrict__ ss_p,
                                                    const int* __restrict__ stop) {
    if (stop && *stop) return;
    const double ua = scalbn(1.0, *det_e - 61), ub = scalbn(1.0, fixed_exp(*ss_p) - 61);
    for (int64_t j = (int64_t)blockIdx.x * 256 + threadIdx.x; j < n; j += (int64_t)gridDim.x * 256) {
        const long long q = ((const long long*)t)[j];
        t[j] = (double)q * (j >= off_instr && j < off_instr + I ? ub : ua);
    }
}

static int instr_copies(const gsr_matrix* A) {
    return ((A->dims.n_instr + 1) / 2 * 16) * NWARP <= 96 * 1024 ? NWARP : 1;
}
static size_t instr_smem(const gsr_matrix* A) {
    return (size_t)((A->dims.n_instr + 1) / 2 * 16) * instr_copies(A);
}

// shared memory of k_aprod2<., ., INSTR = false>: the windows and the y tiles only
static int aprod2_main_smem(const gsr_matrix* A) { return NWARP_MAIN * 3 * A->wstride * 8 + NWARP_MAIN * 32 * 8; }

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
    GSR_TRY(set_smem(k_aprod2<false, false, true>, b));
    GSR_TRY(set_smem(k_aprod2<false, true, true>, b));
    GSR_TRY(set_smem(k_aprod2<true, false, true>, b));
    GSR_TRY(set_smem(k_aprod2<false, false, false>, aprod2_main_smem(A)));
    GSR_TRY(set_smem(k_aprod2<false, true, false>, aprod2_main_smem(A)));
    GSR_TRY(set_smem(k_fused<false>, A->smem_fused));
    GSR_TRY(set_smem(k_fused<true>, A->smem_fused));
    GSR_TRY(set_smem(k_aprod2_instr<false>, (int)instr_smem(A)));
    GSR_TRY(set_smem(k_aprod2_instr<true>, (int)instr_smem(A)));
    {
        int nb = 1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_fused<false>, TPB, A->smem_fused) != cudaSuccess || nb < 1) {
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
    A->grid2 = A->sm_count * resident_ctas(k_aprod2<false, false, true>, A);
    {
        int nb = 1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_aprod2<false, false, false>, NWARP_MAIN * 32, aprod2_main_smem(A)) != cudaSuccess || nb < 1) {
            cudaGetLastError();
            nb = 1;
        }
        A->grid2_main = A->sm_count * nb;
    }
    return GSR_OK;   // (a launch over few units takes fewer CTAs: grid_for)
}

static int reset_counter(const gsr_matrix* A, cudaStream_t s) {
    GSR_CUDA_TRY(cudaMemsetAsync(A->unit_counter, 0, sizeof(int), s));
    return GSR_OK;
}

// persistent grid of a launch over `nu` units: never more CTAs than there are units for
static int grid_for(int grid, int nu) {
    const int need = (nu + NWARP - 1) / NWARP;
    return grid < need ? grid : (need > 0 ? need : 1);
}
// a whole pass = the resident view, or the resident view + the streamed chunks (row f4(iii))
static int pass(const gsr_matrix* A, cudaStream_t s, const std::function<int(const TileView&)>& f) {
    if (!A->so.on) {
        const TileView v{A->tiles, 0, A->n_units, 0, A->n_tiles};
        return f(v);
    }
    return for_each_view(const_cast<gsr_matrix*>(A), s, f);
}

static int aprod1_view(const gsr_matrix* A, const TileView& v, const double* x, double* y, const double* ca,
                       double* partials, const int* stop, const uint32_t* perm, cudaStream_t s) {
    const int nu = v.u1 - v.u0;
    if (nu <= 0) return GSR_OK;
    const int64_t S = A->dims.n_stars, D = A->dims.n_dfa;
    const int I = (int)A->dims.n_instr;
    const int grid = grid_for(A->grid1, nu);
    const Unit* un = A->units + v.u0;
    double* pu = partials ? partials + v.u0 : nullptr;
    GSR_TRY(reset_counter(A, s));
    if (perm)
        k_aprod1<false, true><<<grid, TPB, A->smem_bytes, s>>>(
            v.base, un, nu, A->unit_counter, x, y, ca, nullptr, perm, S, D, I, A->win, A->wstride, stop);
    else if (partials)
        k_aprod1<true, false><<<grid, TPB, A->smem_bytes, s>>>(
            v.base, un, nu, A->unit_counter, x, y, ca, pu, nullptr, S, D, I, A->win, A->wstride, stop);
    else
        k_aprod1<false, false><<<grid, TPB, A->smem_bytes, s>>>(
            v.base, un, nu, A->unit_counter, x, y, ca, nullptr, nullptr, S, D, I, A->win, A->wstride, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_aprod1(const gsr_matrix* A, const double* x, double* y, const double* ca,
                  double* partials, const int* stop, const uint32_t* perm, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    return pass(A, s, [&](const TileView& v) { return aprod1_view(A, v, x, y, ca, partials, stop, perm, s); });
}

// ss != nullptr (the solver's own calls): device sum of y^2 over ALL rows of the product.  On a
// column-scaled matrix the instrumental block is then done by the exact fixed-point pass of the
// fused iteration (reading A22: normwise accuracy, which is what LSQR needs) after a main launch
// without it, instead of six fp64 compare-and-swap adds per row inside the sweep.
static int aprod2_view(const gsr_matrix* A, const TileView& v, const double* y, double* x, const double* sy,
                       const int* stop, const uint32_t* perm, bool square, const double* ss, cudaStream_t s) {
    const int nu = v.u1 - v.u0;
    if (nu <= 0) return GSR_OK;
    const int64_t S = A->dims.n_stars, D = A->dims.n_dfa;
    const int I = (int)A->dims.n_instr;
    const Unit* un = A->units + v.u0;
    GSR_TRY(reset_counter(A, s));
    if (square) {
        k_aprod2<true, false, true><<<grid_for(A->grid2, nu), TPB, A->smem_bytes, s>>>(
            v.base, un, nu, A->unit_counter, nullptr, x, nullptr, nullptr, S, D, I, A->win, A->wstride, instr_copies(A), nullptr, nullptr);
        count_launch();
        GSR_CUDA_TRY(cudaGetLastError());
        return GSR_OK;
    }
    const bool fixed = ss != nullptr && A->p != nullptr && !A->opt_no_fixed && perm == nullptr;
    if (!fixed && !aprod2_is_split(A)) {
        if (perm)
            k_aprod2<false, true, true><<<grid_for(A->grid2, nu), TPB, A->smem_bytes, s>>>(
                v.base, un, nu, A->unit_counter, y, x, sy, perm, S, D, I, A->win, A->wstride, instr_copies(A), stop, nullptr);
        else
            k_aprod2<false, false, true><<<grid_for(A->grid2, nu), TPB, A->smem_bytes, s>>>(
                v.base, un, nu, A->unit_counter, y, x, sy, nullptr, S, D, I, A->win, A->wstride, instr_copies(A), stop, nullptr);
        count_launch();
        GSR_CUDA_TRY(cudaGetLastError());
        return GSR_OK;
    }
    // two launches (default): everything but the instrumental block, then the instrumental pass
    // over the instrumental planes alone (fp64 adds: a caller's y has no norm bound to scale by)
    const int need_main = (nu + NWARP_MAIN - 1) / NWARP_MAIN;
    const int grid = A->grid2_main < need_main ? A->grid2_main : (need_main > 0 ? need_main : 1);
    const int smem = aprod2_main_smem(A);
    const double* yi = y + v.t0 * R;   // internal order: the view's slice of y
    const double* syi = sy;
    if (perm) {
        if (!A->yint) return GSR_ESTATE;
        k_aprod2<false, true, false><<<grid, NWARP_MAIN * 32, smem, s>>>(
            v.base, un, nu, A->unit_counter, y, x, sy, perm, S, D, I, A->win, A->wstride, 1, stop, A->yint);
        yi = A->yint + v.t0 * R;       // already scaled
        syi = nullptr;
    } else {
        k_aprod2<false, false, false><<<grid, NWARP_MAIN * 32, smem, s>>>(
            v.base, un, nu, A->unit_counter, y, x, sy, nullptr, S, D, I, A->win, A->wstride, 1, stop, nullptr);
    }
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    const int64_t nt = v.t1 - v.t0;
    const int64_t need = (nt + NWARP - 1) / NWARP;
    const int gi = A->grid_instr < need ? A->grid_instr : (int)need;
    if (fixed)
        k_aprod2_instr<true><<<gi, TPB, instr_smem(A), s>>>(
            v.base + v.t0 * TILE_BYTES, nt, yi, x + A->off_instr, I, instr_copies(A), ss, stop, 0, syi);
    else
        k_aprod2_instr<false><<<gi, TPB, instr_smem(A), s>>>(
            v.base + v.t0 * TILE_BYTES, nt, yi, x + A->off_instr, I, instr_copies(A), nullptr, stop, 0, syi);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_aprod2(const gsr_matrix* A, const double* y, double* x, const double* sy,
                  const int* stop, const uint32_t* perm, cudaStream_t s, const double* ss) {
    if (A->n_units == 0) return GSR_OK;
    return pass(A, s, [&](const TileView& v) { return aprod2_view(A, v, y, x, sy, stop, perm, false, ss, s); });
}

static int fused_view(const gsr_matrix* A, const TileView& v, const double* x, double* u, const double* ca,
                      double* partials, double* t, const int* stop, const int* det_e, cudaStream_t s) {
    const int nu = v.u1 - v.u0;
    if (nu <= 0) return GSR_OK;
    const int grid = grid_for(A->grid_fused, nu);
    GSR_TRY(reset_counter(A, s));
    if (det_e)
        k_fused<true><<<grid, TPB, A->smem_fused, s>>>(
            v.base, A->units + v.u0, nu, A->unit_counter, x, u, ca, partials + v.u0, t, A->dims.n_stars,
            A->dims.n_dfa, (int)A->dims.n_instr, A->win, A->wstride, stop, det_e);
    else
        k_fused<false><<<grid, TPB, A->smem_fused, s>>>(
            v.base, A->units + v.u0, nu, A->unit_counter, x, u, ca, partials + v.u0, t, A->dims.n_stars,
            A->dims.n_dfa, (int)A->dims.n_instr, A->win, A->wstride, stop, nullptr);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

static int instr_view(const gsr_matrix* A, const TileView& v, const double* u, double* t, const double* ss,
                      const int* stop, int det, bool fixed, cudaStream_t s) {
    const int64_t nt = v.t1 - v.t0;
    if (nt <= 0) return GSR_OK;
    const int64_t need = (nt + NWARP - 1) / NWARP;
    const int grid = A->grid_instr < need ? A->grid_instr : (int)need;
    const unsigned char* T0 = v.base + v.t0 * TILE_BYTES;
    if (fixed)
        k_aprod2_instr<true><<<grid, TPB, instr_smem(A), s>>>(
            T0, nt, u + v.t0 * R, t + A->off_instr, (int)A->dims.n_instr, instr_copies(A), ss, stop, det, nullptr);
    else
        k_aprod2_instr<false><<<grid, TPB, instr_smem(A), s>>>(
            T0, nt, u + v.t0 * R, t + A->off_instr, (int)A->dims.n_instr, instr_copies(A), nullptr, stop, 0, nullptr);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_fused(const gsr_matrix* A, const double* v, double* u, const double* ca,
                 double* partials, double* t, const int* stop, const int* det_e, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    return pass(A, s, [&](const TileView& w) { return fused_view(A, w, v, u, ca, partials, t, stop, det_e, s); });
}

int launch_aprod2_instr(const gsr_matrix* A, const double* u, double* t, const double* ss,
                        const int* stop, int det, cudaStream_t s) {
    if (A->n_tiles == 0) return GSR_OK;
    if (det && (A->p == nullptr || ss == nullptr)) return GSR_ESTATE;
    // exact fixed-point accumulation needs unit column norms (see k_aprod2_instr) and ||u||^2
    const bool fixed = A->p != nullptr && ss != nullptr && (!A->opt_no_fixed || det);
    return pass(A, s, [&](const TileView& w) { return instr_view(A, w, u, t, ss, stop, det, fixed, s); });
}

// Streamed systems: both kernels of the fused iteration on every view while its tiles are on the
// device, so that the host part of the matrix crosses the bus ONCE per iteration.  The
// instrumental pass cannot know ||u_hat|| of the whole pass yet, hence fp64 atomics (the pass
// is bound by the bus, not by them).
int launch_fused_streamed(const gsr_matrix* A, const double* v, double* u, const double* ca,
                          double* partials, double* t, const int* stop, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    return pass(A, s, [&](const TileView& w) {
        GSR_TRY(fused_view(A, w, v, u, ca, partials, t, stop, nullptr, s));
        return instr_view(A, w, u, t, nullptr, stop, 0, false, s);
    });
}

int launch_det_finish(const gsr_matrix* A, double* t, const int* det_e, const double* ss,
                      const int* stop, cudaStream_t s) {
    k_det_finish<<<592, 256, 0, s>>>(t, A->n_cols, A->off_instr, A->dims.n_instr, det_e, ss, stop);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

int launch_colsumsq(const gsr_matrix* A, double* q, cudaStream_t s) {
    if (A->n_units == 0) return GSR_OK;
    return pass(A, s, [&](const TileView& v) { return aprod2_view(A, v, nullptr, q, nullptr, nullptr, nullptr, true, nullptr, s); });
}

// caller row order <-> internal row order of an m-sized vector (gsr_vector_to_internal /
// gsr_vector_from_internal): streaming passes over perm; rows move only inside their ingest
// segment (2^22 rows = 32 MB of doubles), so the scattered side stays in L2
__global__ void __launch_bounds__(256) k_rows_to_internal(const double* __restrict__ src,
                                                          const uint32_t* __restrict__ perm,
                                                          double* __restrict__ dst, int64_t len_int) {
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < len_int; i += (int64_t)gridDim.x * 256) {
        const uint32_t pe = perm[i];
        dst[i] = pe != PERM_PAD ? src[pe] : 0.0;     // padding rows of a tile hold zero
    }
}
__global__ void __launch_bounds__(256) k_rows_from_internal(const double* __restrict__ src,
                                                            const uint32_t* __restrict__ perm,
                                                            double* __restrict__ dst, int64_t len_int) {
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < len_int; i += (int64_t)gridDim.x * 256) {
        const uint32_t pe = perm[i];
        if (pe != PERM_PAD) dst[pe] = src[i];
    }
}

}  // namespace gsr

using namespace gsr;

extern "C" {

int64_t gsr_matrix_internal_rows(const gsr_matrix* A) { return (A && A->state == 1) ? A->m_int + A->n_con : -1; }

int gsr_vector_to_internal(const gsr_matrix* A, const double* y_dev, double* yint_dev, gsr_stream stream) {
    if (!A || ((!y_dev || !yint_dev) && A->dims.n_rows + A->n_con > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    cudaStream_t s = (cudaStream_t)stream;
    if (A->m_int > 0) {
        k_rows_to_internal<<<A->sm_count * 8, 256, 0, s>>>(y_dev, A->perm, yint_dev, A->m_int);
        count_launch();
        GSR_CUDA_TRY(cudaGetLastError());
    }
    if (A->n_con > 0)   // constraint rows keep their order, after the observations
        GSR_CUDA_TRY(cudaMemcpyAsync(yint_dev + A->m_int, y_dev + A->dims.n_rows, (size_t)A->n_con * 8,
                                     cudaMemcpyDeviceToDevice, s));
    return GSR_OK;
}

int gsr_vector_from_internal(const gsr_matrix* A, const double* yint_dev, double* y_dev, gsr_stream stream) {
    if (!A || ((!y_dev || !yint_dev) && A->dims.n_rows + A->n_con > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    cudaStream_t s = (cudaStream_t)stream;
    if (A->m_int > 0) {
        k_rows_from_internal<<<A->sm_count * 8, 256, 0, s>>>(yint_dev, A->perm, y_dev, A->m_int);
        count_launch();
        GSR_CUDA_TRY(cudaGetLastError());
    }
    if (A->n_con > 0)
        GSR_CUDA_TRY(cudaMemcpyAsync(y_dev + A->dims.n_rows, yint_dev + A->m_int, (size_t)A->n_con * 8,
                                     cudaMemcpyDeviceToDevice, s));
    return GSR_OK;
}

int gsr_aprod1_internal(const gsr_matrix* A, const double* x_dev, double* yint_dev, gsr_stream stream) {
    if (!A || !x_dev || (!yint_dev && A->m_int + A->n_con > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    GSR_TRY(launch_aprod1(A, x_dev, yint_dev, A->coef_one, nullptr, nullptr, nullptr, (cudaStream_t)stream));
    return launch_con_aprod1(A, x_dev, yint_dev + A->m_int, A->coef_one, nullptr, nullptr, (cudaStream_t)stream);
}

int gsr_aprod2_internal(const gsr_matrix* A, const double* yint_dev, double* x_dev, gsr_stream stream) {
    if (!A || !x_dev || (!yint_dev && A->m_int + A->n_con > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    GSR_TRY(launch_aprod2(A, yint_dev, x_dev, A->coef_one, nullptr, nullptr, (cudaStream_t)stream));
    return launch_con_aprod2(A, yint_dev + A->m_int, x_dev, A->coef_one, nullptr, (cudaStream_t)stream);
}

int gsr_aprod1(const gsr_matrix* A, const double* x_dev, double* y_dev, gsr_stream stream) {
    if (!A || !x_dev || (!y_dev && A->dims.n_rows > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    GSR_TRY(launch_aprod1(A, x_dev, y_dev, A->coef_one, nullptr, nullptr, A->perm, (cudaStream_t)stream));
    return launch_con_aprod1(A, x_dev, y_dev + A->dims.n_rows, A->coef_one, nullptr, nullptr, (cudaStream_t)stream);
}

int gsr_aprod2(const gsr_matrix* A, const double* y_dev, double* x_dev, gsr_stream stream) {
    if (!A || !x_dev || (!y_dev && A->dims.n_rows > 0)) return GSR_EINVAL;
    if (A->state != 1) return GSR_ESTATE;
    if (aprod2_is_split(A) && !A->yint && A->m_int > 0) {
        // scratch of the split form (a cache behind a logically const handle): y in internal order
        gsr_matrix* Am = const_cast<gsr_matrix*>(A);
        GSR_TRY(dev_alloc(Am, (void**)&Am->yint, (size_t)A->m_int * 8));
    }
    GSR_TRY(launch_aprod2(A, y_dev, x_dev, A->coef_one, nullptr, A->perm, (cudaStream_t)stream));
    return launch_con_aprod2(A, y_dev + A->dims.n_rows, x_dev, A->coef_one, nullptr, (cudaStream_t)stream);
}

}  // extern "C"
