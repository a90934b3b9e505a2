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

void dev_free(gsr_matrix* A, void* p, size_t bytes) {
    if (!p) return;
    cudaFree(p);
    A->device_bytes -= (int64_t)(bytes == 0 ? 8 : bytes);
}

// ---- segment partition: stable counting sort of the staged rows by fine attitude bin ------
constexpr int BLK = 1024;   // staged rows per block of the partition kernels

// Pass 1: per block of BLK staged rows, rows per bin -> counts[bin * nblk + blk]; validation.
// Error bits: 1 star out of range, 2 star decreasing, 4 att_start out of range, 8 instr_col.
__global__ void __launch_bounds__(BLK) k_seg_count(const int32_t* __restrict__ star,
                                                   const int32_t* __restrict__ att,
                                                   const int32_t* __restrict__ instr, int64_t ns,
                                                   int64_t S, int64_t D, int64_t I, int bin_width,
                                                   int nbins, int nblk, int* __restrict__ counts,
                                                   const int* __restrict__ last_star,
                                                   int* __restrict__ err) {
    extern __shared__ int hist[];
    for (int b = threadIdx.x; b < nbins; b += BLK) hist[b] = 0;
    __syncthreads();
    const int64_t r = (int64_t)blockIdx.x * BLK + threadIdx.x;
    if (r < ns) {
        int e = 0;
        const int32_t s = star[r], a = att[r];
        if (s < 0 || s >= S) e |= 1;
        const int32_t sprev = r > 0 ? star[r - 1] : *last_star;
        if (s < sprev) e |= 2;
        int bin = 0;
        if (a < 0 || a > D - 4) e |= 4;
        else bin = a / bin_width;
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const int32_t c = instr[6 * r + j];
            if (c < 0 || c >= I) e |= 8;
        }
        if (e) atomicOr(err, e);
        atomicAdd(&hist[bin], 1);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins; b += BLK) counts[(int64_t)b * nblk + blockIdx.x] = hist[b];
}

// Pass 2 (one CTA): exclusive scan of counts in (bin, block) order; every bin starts on a tile
// boundary.  counts[] becomes the destination offset (rows from the segment's first tile);
// bin_info[b] = rows in bin b, bin_info[nbins + b] = padded start row of bin b,
// bin_info[2*nbins] = padded rows of the whole segment.
__global__ void __launch_bounds__(1024) k_seg_scan(int* __restrict__ counts, int nbins, int nblk,
                                                   int* __restrict__ bin_info) {
    __shared__ int part[1024];
    __shared__ int wsum[32];
    int base = 0;
    const int per = (nblk + 1023) / 1024;
    const int i0 = threadIdx.x * per, i1 = min(i0 + per, nblk);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int b = 0; b < nbins; ++b) {
        int* c = counts + (int64_t)b * nblk;
        int s = 0;
        for (int i = i0; i < i1; ++i) s += c[i];
        // exclusive scan of the 1024 per-thread sums
        int incl = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int up = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += up;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int w = wsum[lane], wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int up = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += up;
            }
            wsum[lane] = wi - w;           // exclusive warp offsets
            if (lane == 31) part[0] = wi;  // total rows of the bin
        }
        __syncthreads();
        const int run = part[0];
        int off = base + wsum[warp] + incl - s;
        for (int i = i0; i < i1; ++i) {
            const int v = c[i];
            c[i] = off;
            off += v;
        }
        if (threadIdx.x == 0) {
            bin_info[b] = run;
            bin_info[nbins + b] = base;
        }
        base += ((run + R - 1) / R) * R;
        __syncthreads();
    }
    if (threadIdx.x == 0) bin_info[2 * nbins] = base;
}

// Pass 3: stable scatter of the staged rows into tile records (internal order) + perm.
__global__ void __launch_bounds__(BLK) k_seg_scatter(
    unsigned char* __restrict__ tiles, uint32_t* __restrict__ perm, int64_t row_base_int,
    int64_t row_base_ext, const int32_t* __restrict__ star, const int32_t* __restrict__ att,
    const int32_t* __restrict__ instr, const double* __restrict__ vals, int64_t ns, int64_t D,
    int bin_width, int nblk, const int* __restrict__ offs) {
    __shared__ int sbin[BLK];
    const int64_t r = (int64_t)blockIdx.x * BLK + threadIdx.x;
    int bin = -1;
    int32_t a = 0;
    if (r < ns) {
        a = att[r];
        bin = (a >= 0 && a <= D - 4) ? a / bin_width : 0;
    }
    sbin[threadIdx.x] = bin;
    __syncthreads();
    if (r >= ns) return;
    int rank = 0;   // rows of my bin that precede me in this block (stable)
    for (int i = 0; i < (int)threadIdx.x; ++i) rank += sbin[i] == bin;
    const int64_t dst = row_base_int + offs[(int64_t)bin * nblk + blockIdx.x] + rank;
    unsigned char* T = tiles + (dst / R) * (int64_t)TILE_BYTES;
    const int lr = (int)(dst % R);
    perm[dst] = (uint32_t)(row_base_ext + r);
    ((int32_t*)(T + OFF_STAR))[lr] = star[r];
    const int a0 = bin * bin_width;
    (T + OFF_AOFF)[att_slot(lr)] = (unsigned char)(bin == 0 && (a < 0 || a > D - 4) ? 0 : a - a0);
    *(int32_t*)(T + OFF_A0) = a0;   // same value from every row of the tile
#pragma unroll
    for (int j = 0; j < 6; ++j) *(uint16_t*)(T + icol_offset(j, lr)) = (uint16_t)instr[6 * r + j];
#pragma unroll
    for (int k = 0; k < NPAR; ++k) *(double*)(T + val_offset(k, lr)) = vals[NPAR * r + k];
}

__global__ void k_save_last_star(const int32_t* __restrict__ star, int64_t ns, int* last_star) {
    if (ns > 0) *last_star = star[ns - 1];
}

// Padding rows (they round every bin up to whole tiles and trail the bin's real rows): zero
// coefficients, window offset 0 and instrumental column 0 (tiles are memset to 0); star = the
// star of the last real row of the tile, so that they open no new star segment.  Also writes
// the tile's overlap mask: bit q is set when the windows of attitude slots (0, q) and (1, q)
// overlap, i.e. when aprod2 must not add the two in one instruction.
// One warp per tile.
__global__ void __launch_bounds__(256) k_fix_padding(unsigned char* __restrict__ tiles,
                                                     const uint32_t* __restrict__ perm,
                                                     int64_t t_begin, int64_t n_tiles) {
    int64_t t = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (t >= n_tiles) return;
    t += t_begin;
    const int lane = threadIdx.x & 31;
    unsigned char* T = tiles + t * TILE_BYTES;
    const bool real = perm[t * R + lane] != PERM_PAD;
    const int nreal = __popc(__ballot_sync(0xffffffffu, real));
    if (!real) ((int32_t*)(T + OFF_STAR))[lane] = nreal > 0 ? ((const int32_t*)(T + OFF_STAR))[nreal - 1] : 0;
    const int da = (int)(T + OFF_AOFF)[lane & 15] - (int)(T + OFF_AOFF)[16 + (lane & 15)];
    const unsigned cmask = __ballot_sync(0xffffffffu, lane < 16 && da > -4 && da < 4);
    if (lane == 0) *(uint32_t*)(T + OFF_CMASK) = cmask;
}

// Bank spreading of the instrumental block.  The six (column, value) pairs of a row may sit in
// any of the six slots, and the product kernels gather / scatter slot by slot with the 16 home
// lanes of a half-warp in one shared-memory wavefront group: 16 random columns fall into the 16
// eight-byte banks with a maximum load of about 3.1, i.e. 6 wavefronts per 32-lane access
// instead of 2.  A greedy pass per half-warp (rows in order; the entry whose bank is most loaded
// so far first; into the free slot where that bank is least loaded) brings the six accesses of
// a half from 18.5 to 12.4 wavefronts on uniform columns.  One thread per (tile, half).
__global__ void __launch_bounds__(128) k_permute_instr(unsigned char* __restrict__ tiles,
                                                       const uint32_t* __restrict__ perm,
                                                       int64_t t_begin, int64_t n_tiles) {
    const int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= 2 * n_tiles) return;
    const int64_t t = t_begin + (id >> 1);
    const int l0 = (int)(id & 1) * 16;
    unsigned char* T = tiles + t * TILE_BYTES;
    unsigned char cnt[6][16];
    for (int k = 0; k < 6; ++k)
        for (int b = 0; b < 16; ++b) cnt[k][b] = 0;
    for (int r = 0; r < 16; ++r) {
        const int lr = l0 + r;
        if (perm[t * R + lr] == PERM_PAD) {   // zero rows keep column 0 in every slot
            *(uint16_t*)(T + OFF_IPERM + lr * 2) = (uint16_t)(0 + 1 * 6 + 2 * 36 + 3 * 216 + 4 * 1296 + 5 * 7776);
            continue;
        }
        uint16_t c[6];
        double v[6];
        int tot[6];
        for (int e = 0; e < 6; ++e) {
            c[e] = *(const uint16_t*)(T + icol_offset(e, lr));
            v[e] = *(const double*)(T + val_offset(17 + e, lr));
            int s = 0;
            for (int k = 0; k < 6; ++k) s += cnt[k][c[e] & 15];
            tot[e] = s;
        }
        unsigned done = 0, used = 0;
        int code = 0, pow6 = 1;
        int slot_of[6];
        for (int step = 0; step < 6; ++step) {
            int be = -1;
            for (int e = 0; e < 6; ++e)
                if (!((done >> e) & 1u) && (be < 0 || tot[e] > tot[be])) be = e;
            const int b = c[be] & 15;
            int bk = -1;
            for (int k = 0; k < 6; ++k)
                if (!((used >> k) & 1u) && (bk < 0 || cnt[k][b] < cnt[bk][b])) bk = k;
            done |= 1u << be;
            used |= 1u << bk;
            cnt[bk][b]++;
            slot_of[be] = bk;
        }
        for (int e = 0; e < 6; ++e) {
            *(uint16_t*)(T + icol_offset(slot_of[e], lr)) = c[e];
            *(double*)(T + val_offset(17 + slot_of[e], lr)) = v[e];
            code += slot_of[e] * pow6;
            pow6 *= 6;
        }
        *(uint16_t*)(T + OFF_IPERM + lr * 2) = (uint16_t)code;
    }
}

// Caller-order dump of rows [row0, row0+nrows): every internal row whose caller row falls in
// the range writes its 24 (column, value) pairs.
__global__ void k_expand_rows(const unsigned char* __restrict__ tiles, const uint32_t* __restrict__ perm,
                              int64_t r_begin, int64_t r_end, int64_t row0, int64_t nrows, int64_t S, int64_t D,
                              int64_t I, int64_t* __restrict__ cols, double* __restrict__ vals) {
    const int64_t ri = r_begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (ri >= r_end) return;
    const uint32_t pe = perm[ri];
    if (pe == PERM_PAD) return;
    const int64_t r = (int64_t)pe - row0;
    if (r < 0 || r >= nrows) return;
    const unsigned char* T = tiles + (ri / R) * (int64_t)TILE_BYTES;
    const int lr = (int)(ri % R);
    const int64_t s = ((const int32_t*)(T + OFF_STAR))[lr];
    const int64_t a = (int64_t)(*(const int32_t*)(T + OFF_A0)) + (T + OFF_AOFF)[att_slot(lr)];
    const int64_t off_att = 5 * S, off_instr = off_att + 3 * D, off_glob = off_instr + I;
    int slot[6];   // slot of the caller's e-th instrumental entry (k_permute_instr)
    int code = *(const uint16_t*)(T + OFF_IPERM + lr * 2);
    for (int e = 0; e < 6; ++e) {
        slot[e] = code % 6;
        code /= 6;
    }
    for (int k = 0; k < NPAR; ++k) {
        int64_t c;
        if (k < 5) c = 5 * s + k;
        else if (k < 17) c = off_att + ((k - 5) / 4) * D + a + (k - 5) % 4;
        else if (k < 23) c = off_instr + *(const uint16_t*)(T + icol_offset(slot[k - 17], lr));
        else c = off_glob;
        cols[NPAR * r + k] = c;
        vals[NPAR * r + k] = *(const double*)(T + val_offset(k >= 17 && k < 23 ? 17 + slot[k - 17] : k, lr));
    }
}

// p_j = q_j > 0 ? 1/sqrt(q_j) : 1   (reading A7)
__global__ void k_make_p(double* __restrict__ p, int64_t n) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    double q = p[j];
    p[j] = q > 0.0 ? 1.0 / sqrt(q) : 1.0;
}

// values[i,k] *= p[col(i,k)] in place, one thread per row (8 tiles per CTA).
__global__ void __launch_bounds__(256) k_scale_values(unsigned char* __restrict__ tiles,
                                                      int64_t t_begin, int64_t n_tiles,
                                                      const double* __restrict__ p,
                                                      int64_t S, int64_t D, int64_t I) {
    const int64_t t = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (t >= n_tiles) return;
    unsigned char* T = tiles + (t_begin + t) * TILE_BYTES;
    const int lr = threadIdx.x & 31;
    const int64_t s = ((const int32_t*)(T + OFF_STAR))[lr];
    const int64_t a = (int64_t)(*(const int32_t*)(T + OFF_A0)) + (T + OFF_AOFF)[att_slot(lr)];
    const double* pa = p + 5 * s;
    const double* pt = p + 5 * S + a;
    const double* pi = p + 5 * S + 3 * D;
#pragma unroll
    for (int k = 0; k < 5; ++k) *(double*)(T + val_offset(k, lr)) *= pa[k];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax)
#pragma unroll
        for (int j = 0; j < 4; ++j) *(double*)(T + val_offset(5 + 4 * ax + j, lr)) *= pt[ax * D + j];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const int c = *(const uint16_t*)(T + icol_offset(j, lr));
        *(double*)(T + val_offset(17 + j, lr)) *= pi[c];
    }
    *(double*)(T + val_offset(23, lr)) *= pi[I];
}

// ---- out-of-core passes (row f4(iii)) -----------------------------------------------------
// Copy chunk c into buffer c & 1 on the copy stream, as soon as the buffer's last consumer
// (event done[b], recorded on the compute stream) has finished.  Tiles below res_cap come from
// the device array (only the first chunk can straddle the boundary), the rest from the host.
static int issue_chunk_copy(gsr_matrix* A, size_t c) {
    StreamStore& so = A->so;
    const Chunk& ch = (*so.chunks)[c];
    const int b = (int)(c & 1);
    GSR_CUDA_TRY(cudaStreamWaitEvent(so.copy, so.done[b], 0));
    const int64_t td = ch.t1 < so.res_cap ? ch.t1 : so.res_cap;
    if (ch.t0 < td)
        GSR_CUDA_TRY(cudaMemcpyAsync(so.buf[b], A->tiles + ch.t0 * TILE_BYTES, (size_t)(td - ch.t0) * TILE_BYTES,
                                     cudaMemcpyDeviceToDevice, so.copy));
    const int64_t th = ch.t0 > so.res_cap ? ch.t0 : so.res_cap;
    if (th < ch.t1) {
        GSR_CUDA_TRY(cudaMemcpyAsync(so.buf[b] + (th - ch.t0) * TILE_BYTES, so.host + (th - so.res_cap) * TILE_BYTES,
                                     (size_t)(ch.t1 - th) * TILE_BYTES, cudaMemcpyHostToDevice, so.copy));
        so.h2d_bytes += (ch.t1 - th) * TILE_BYTES;
    }
    GSR_CUDA_TRY(cudaEventRecord(so.copied[b], so.copy));
    return GSR_OK;
}

int for_each_view(gsr_matrix* A, cudaStream_t s, const std::function<int(const TileView&)>& f, bool writeback) {
    StreamStore& so = A->so;
    const std::vector<Chunk>& chunks = *so.chunks;
    const size_t nc = chunks.size();
    // After ingest or a write-back pass the copy stream starts after whatever has been queued on s
    // so far (the tiles it reads were written there).  After a read-only pass nothing it reads can
    // change: the copies only wait for their buffer (done[b]) and run ahead of the kernels by up to
    // two chunks -- across the end of the previous pass too.
    if (so.need_fork) {
        GSR_CUDA_TRY(cudaEventRecord(so.fork, s));
        GSR_CUDA_TRY(cudaStreamWaitEvent(so.copy, so.fork, 0));
        so.need_fork = false;
    }
    for (size_t c = 0; c < nc && c < 2; ++c) GSR_TRY(issue_chunk_copy(A, c));
    if (so.res_units > 0) {
        const Unit& last = (*A->units_host)[so.res_units - 1];
        const TileView v{A->tiles, 0, so.res_units, 0, (int64_t)last.tile0 + last.ntiles};
        GSR_TRY(f(v));
    }
    for (size_t c = 0; c < nc; ++c) {
        const Chunk& ch = chunks[c];
        const int b = (int)(c & 1);
        GSR_CUDA_TRY(cudaStreamWaitEvent(s, so.copied[b], 0));
        const TileView v{so.buf[b] - ch.t0 * TILE_BYTES, ch.u0, ch.u1, ch.t0, ch.t1};
        GSR_TRY(f(v));
        if (writeback) {
            const int64_t td = ch.t1 < so.res_cap ? ch.t1 : so.res_cap;
            if (ch.t0 < td)
                GSR_CUDA_TRY(cudaMemcpyAsync(A->tiles + ch.t0 * TILE_BYTES, so.buf[b], (size_t)(td - ch.t0) * TILE_BYTES,
                                             cudaMemcpyDeviceToDevice, s));
            const int64_t th = ch.t0 > so.res_cap ? ch.t0 : so.res_cap;
            if (th < ch.t1)
                GSR_CUDA_TRY(cudaMemcpyAsync(so.host + (th - so.res_cap) * TILE_BYTES, so.buf[b] + (th - ch.t0) * TILE_BYTES,
                                             (size_t)(ch.t1 - th) * TILE_BYTES, cudaMemcpyDeviceToHost, s));
        }
        GSR_CUDA_TRY(cudaEventRecord(so.done[b], s));
        if (c + 2 < nc) GSR_TRY(issue_chunk_copy(A, c + 2));
    }
    if (writeback) so.need_fork = true;
    return GSR_OK;
}

void free_stream_store(gsr_matrix* A) {
    StreamStore& so = A->so;
    if (so.host) cudaFreeHost(so.host);
    for (int b = 0; b < 2; ++b) {
        if (so.buf[b]) dev_free(A, so.buf[b], (size_t)so.chunk_cap * TILE_BYTES);
        if (so.copied[b]) cudaEventDestroy(so.copied[b]);
        if (so.done[b]) cudaEventDestroy(so.done[b]);
    }
    if (so.seg) dev_free(A, so.seg, (size_t)so.seg_cap * TILE_BYTES);
    if (so.fork) cudaEventDestroy(so.fork);
    if (so.copy) cudaStreamDestroy(so.copy);
    delete so.chunks;
    cudaGetLastError();
    so = StreamStore();
}

}  // namespace gsr

using namespace gsr;

// padding rows, overlap masks and bank spreading of tiles [t0, t0 + nt) (base: address of tile 0)
static int finish_tiles(gsr_matrix* A, unsigned char* base, int64_t t0, int64_t nt) {
    if (nt <= 0) return GSR_OK;
    k_fix_padding<<<(unsigned)((nt + 7) / 8), 256, 0, A->stream>>>(base, A->perm, t0, nt);
    k_permute_instr<<<(unsigned)((2 * nt + 127) / 128), 128, 0, A->stream>>>(base, A->perm, t0, nt);
    count_launch(2);
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}

static int flush_segment(gsr_matrix* A) {
    const int64_t ns = A->seg_fill;
    if (ns == 0) return GSR_OK;
    const int nblk = (int)((ns + BLK - 1) / BLK);
    cudaStream_t s = A->stream;
    k_seg_count<<<nblk, BLK, A->nbins * sizeof(int), s>>>(A->st_star, A->st_att, A->st_instr, ns,
                                                        A->dims.n_stars, A->dims.n_dfa, A->dims.n_instr,
                                                        A->bin_width, A->nbins, nblk, A->seg_counts,
                                                        A->last_star, A->err);
    k_seg_scan<<<1, 1024, 0, s>>>(A->seg_counts, A->nbins, nblk, A->seg_bin_rows);
    // out-of-core: the segment's tiles are built in a device buffer of their own and then moved
    // to where they live (device array below res_cap, pinned host memory above)
    unsigned char* base = A->tiles;
    if (A->so.on) {
        GSR_CUDA_TRY(cudaMemsetAsync(A->so.seg, 0, (size_t)A->so.seg_cap * TILE_BYTES, s));
        base = A->so.seg - A->n_tiles * TILE_BYTES;
    }
    k_seg_scatter<<<nblk, BLK, 0, s>>>(base, A->perm, A->n_tiles * R, A->rows_appended - ns,
                                       A->st_star, A->st_att, A->st_instr, A->st_vals, ns,
                                       A->dims.n_dfa, A->bin_width, nblk, A->seg_counts);
    k_save_last_star<<<1, 1, 0, s>>>(A->st_star, ns, A->last_star);
    count_launch(4);
    GSR_CUDA_TRY(cudaGetLastError());
    std::vector<int> info(2 * A->nbins + 1);
    GSR_CUDA_TRY(cudaMemcpyAsync(info.data(), A->seg_bin_rows, info.size() * sizeof(int),
                                 cudaMemcpyDeviceToHost, s));
    GSR_CUDA_TRY(cudaStreamSynchronize(s));
    // unit table: runs of at most unit_tiles tiles inside one (segment, bin); sized so that
    // every resident warp gets several units (dynamic fetch balances the rest)
    const int64_t est_tiles = (A->dims.n_rows + R - 1) / R;
    const int64_t warps = (int64_t)A->sm_count * A->ctas_per_sm * NWARP;
    int64_t unit_tiles = est_tiles / (warps * 8);
    if (unit_tiles < 4) unit_tiles = 4;
    if (unit_tiles > UNIT_TILES_MAX) unit_tiles = UNIT_TILES_MAX;
    for (int b = 0; b < A->nbins; ++b) {
        const int rows = info[b];
        if (rows == 0) continue;
        const int64_t t0 = A->n_tiles + info[A->nbins + b] / R;
        const int64_t nt = (rows + R - 1) / R;
        for (int64_t t = 0; t < nt; t += unit_tiles) {
            Unit u;
            u.tile0 = (int32_t)(t0 + t);
            u.ntiles = (int32_t)(nt - t < unit_tiles ? nt - t : unit_tiles);
            u.a0 = b * A->bin_width;
            u.pad_ = 0;
            A->units_host->push_back(u);
        }
    }
    const int64_t nt_seg = info[2 * A->nbins] / R;
    if (A->n_tiles + nt_seg > A->tiles_cap) return GSR_ECUDA;   // cannot happen: capacity is an upper bound
    if (A->so.on) {
        StreamStore& so = A->so;
        if (nt_seg > so.seg_cap) return GSR_ECUDA;
        GSR_TRY(finish_tiles(A, base, A->n_tiles, nt_seg));
        const int64_t t0 = A->n_tiles, t1 = t0 + nt_seg;
        const int64_t td = t1 < so.res_cap ? t1 : so.res_cap;
        if (t0 < td)
            GSR_CUDA_TRY(cudaMemcpyAsync(A->tiles + t0 * TILE_BYTES, so.seg, (size_t)(td - t0) * TILE_BYTES,
                                         cudaMemcpyDeviceToDevice, s));
        const int64_t th = t0 > so.res_cap ? t0 : so.res_cap;
        if (th < t1)
            GSR_CUDA_TRY(cudaMemcpyAsync(so.host + (th - so.res_cap) * TILE_BYTES, so.seg + (th - t0) * TILE_BYTES,
                                         (size_t)(t1 - th) * TILE_BYTES, cudaMemcpyDeviceToHost, s));
        GSR_CUDA_TRY(cudaStreamSynchronize(s));
    }
    A->n_tiles += nt_seg;
    A->seg_fill = 0;
    return GSR_OK;
}

static void free_staging(gsr_matrix* A) {
    const size_t c = (size_t)A->seg_cap;
    dev_free(A, A->st_star, c * 4); A->st_star = nullptr;
    dev_free(A, A->st_att, c * 4); A->st_att = nullptr;
    dev_free(A, A->st_instr, c * 24); A->st_instr = nullptr;
    dev_free(A, A->st_vals, c * 192); A->st_vals = nullptr;
    if (A->seg_counts) {
        const size_t nblk = (c + BLK - 1) / BLK;
        dev_free(A, A->seg_counts, (size_t)A->nbins * nblk * 4);
        A->seg_counts = nullptr;
    }
}

extern "C" {

const char* gsr_strerror(int code) {
    switch (code) {
        case GSR_OK: return "ok";
        case GSR_EINVAL: return "invalid argument (null pointer, bad dims or index out of range)";
        case GSR_ENOMEM: return "out of device memory";
        case GSR_ECUDA: return "CUDA runtime error";
        case GSR_ESTATE: return "call not legal in this state";
        case GSR_EUNSUPPORTED: return "unsupported device (needs sm_100), size or option";
        case GSR_ERANGE: return "deterministic mode: a pass left the range of its fixed-point sums";
        default: return "unknown gsr status";
    }
}

int64_t gsr_launch_count(void) { return g_launches; }

// resident_bytes < 0: everything on the device.  Otherwise at most resident_bytes of tile storage
// stay on the device and the rest goes to pinned host memory (row f4(iii)).
static int begin_impl(gsr_matrix** out, const gsr_dims* d, gsr_stream stream, int64_t resident_bytes,
                      int64_t chunk_bytes) {
    if (!out) return GSR_EINVAL;
    *out = nullptr;
    if (!d) return GSR_EINVAL;
    if (d->n_rows < 0 || d->n_stars < 1 || d->n_dfa < 4 || d->n_instr < 1 || d->n_glob != 1)
        return GSR_EINVAL;
    const int64_t n = 5 * d->n_stars + 3 * d->n_dfa + d->n_instr + 1;
    if (n >= (int64_t)1 << 31 || d->n_rows >= (int64_t)0xFFFFFFF0) return GSR_EINVAL;
    // shared-memory plan of the product kernels: the whole instrumental block, shared by the
    // warps of a CTA, + one private attitude window of `win` knots x 3 axes per warp
    const int64_t instr_bytes = (d->n_instr + 1) / 2 * 16;
    if (d->n_instr > 65535 || instr_bytes > SMEM_BUDGET - NWARP * 24 * 4) return GSR_EUNSUPPORTED;
    // (the fused iteration kernel keeps two windows per warp: v to read, A^T u to accumulate)
    int64_t win_bytes = (SMEM_BUDGET - instr_bytes - NWARP * 48 * 8) / NWARP / 2;
    if (win_bytes > WIN_BYTES_MAX) win_bytes = WIN_BYTES_MAX;
    const int64_t n_start = d->n_dfa - 3;
    int64_t ws_max = win_bytes / 24;                       // doubles per axis
    ws_max = ws_max - ((ws_max - 4) % 16 + 16) % 16;       // largest value = 4 (mod 16)
    const int64_t bw_max = ws_max - 3;
    if (bw_max < 1) return GSR_EUNSUPPORTED;
    const int64_t nbins = (n_start + bw_max - 1) / bw_max;
    if (nbins > NBIN_MAX) return GSR_EUNSUPPORTED;
    const int64_t bw = (n_start + nbins - 1) / nbins;
    const int64_t wstride = (bw + 3) + ((4 - (bw + 3)) % 16 + 16) % 16;   // >= bw+3, = 4 (mod 16)
    const int64_t instr_copies = instr_bytes * NWARP <= 96 * 1024 ? NWARP : 1;   // as in gsr_aprod.cu
    const int64_t smem_bytes = instr_bytes * instr_copies + NWARP * 3 * wstride * 8 + NWARP * 32 * 8;

    int dev = 0;
    cudaDeviceProp prop;
    GSR_CUDA_TRY(cudaGetDevice(&dev));
    GSR_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return GSR_EUNSUPPORTED;
    gsr_matrix* A = new (std::nothrow) gsr_matrix();
    if (!A) return GSR_ENOMEM;
    memset((void*)A, 0, sizeof(*A));
    new (&A->ws) Workspace();
    A->units_host = new (std::nothrow) std::vector<Unit>();
    A->dims = *d;
    A->n_cols = n;
    A->off_att = 5 * d->n_stars;
    A->off_instr = A->off_att + 3 * d->n_dfa;
    A->off_glob = A->off_instr + d->n_instr;
    A->nbins = (int)nbins;
    A->bin_width = (int)bw;
    A->win = (int)bw + 3;
    A->wstride = (int)wstride;
    A->smem_bytes = (int)smem_bytes;
    A->smem_fused = (int)(instr_bytes + NWARP * 6 * wstride * 8 + NWARP * 48 * 8);
    A->ctas_per_sm = 2 * (smem_bytes + 2048) <= 227 * 1024 ? 2 : 1;
    A->stream = (cudaStream_t)stream;
    A->sm_count = prop.multiProcessorCount;
    A->seg_cap = d->n_rows < SEG ? (d->n_rows > 0 ? d->n_rows : 1) : SEG;
    const int64_t n_seg = (d->n_rows + SEG - 1) / SEG;
    A->tiles_cap = (d->n_rows + R - 1) / R + n_seg * nbins + 1;
    const size_t c = (size_t)A->seg_cap, nblk = (c + BLK - 1) / BLK;
    int64_t dev_tiles = A->tiles_cap;
    int rc = GSR_OK;
    if (resident_bytes >= 0 && resident_bytes / TILE_BYTES < A->tiles_cap) {
        StreamStore& so = A->so;
        so.on = true;
        so.res_cap = resident_bytes / TILE_BYTES;
        so.chunk_cap = chunk_bytes / TILE_BYTES;
        if (so.chunk_cap < 2 * UNIT_TILES_MAX) so.chunk_cap = 2 * UNIT_TILES_MAX;   // a unit always fits
        so.host_cap = A->tiles_cap - so.res_cap;
        so.seg_cap = (A->seg_cap + R - 1) / R + nbins + 1;
        so.chunks = new (std::nothrow) std::vector<Chunk>();
        dev_tiles = so.res_cap > 0 ? so.res_cap : 1;
        if (!so.chunks || cudaHostAlloc((void**)&so.host, (size_t)so.host_cap * TILE_BYTES, cudaHostAllocDefault) != cudaSuccess) {
            cudaGetLastError();
            so.host = nullptr;
            rc = GSR_ENOMEM;
        }
        if (rc == GSR_OK) rc = dev_alloc(A, (void**)&so.seg, (size_t)so.seg_cap * TILE_BYTES);
    }
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->tiles, (size_t)dev_tiles * TILE_BYTES);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->perm, (size_t)A->tiles_cap * R * 4);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->st_star, c * 4);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->st_att, c * 4);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->st_instr, c * 24);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->st_vals, c * 192);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->seg_counts, (size_t)nbins * nblk * 4);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->seg_bin_rows, (2 * nbins + 1) * 4);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->last_star, 4);
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->err, sizeof(int));
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->coef_one, 2 * sizeof(double));
    if (rc == GSR_OK) rc = dev_alloc(A, (void**)&A->unit_counter, sizeof(int));
    if (rc != GSR_OK || !A->units_host) {
        gsr_matrix_destroy(A);
        return rc != GSR_OK ? rc : GSR_ENOMEM;
    }
    const double ones[2] = {1.0, 1.0};
    cudaError_t e = cudaMemsetAsync(A->tiles, 0, (size_t)dev_tiles * TILE_BYTES, A->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A->perm, 0xFF, (size_t)A->tiles_cap * R * 4, A->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A->err, 0, sizeof(int), A->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A->last_star, 0, 4, A->stream);
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

int gsr_matrix_begin(gsr_matrix** out, const gsr_dims* d, gsr_stream stream) {
    return begin_impl(out, d, stream, -1, 0);
}

int gsr_matrix_begin_streamed(gsr_matrix** out, const gsr_dims* d, int64_t resident_bytes,
                              int64_t chunk_bytes, gsr_stream stream) {
    if (resident_bytes < 0 || chunk_bytes < 0) {
        if (out) *out = nullptr;
        return GSR_EINVAL;
    }
    return begin_impl(out, d, stream, resident_bytes, chunk_bytes);
}

int64_t gsr_matrix_host_bytes(const gsr_matrix* A) {
    return (A && A->so.on) ? A->so.host_cap * (int64_t)TILE_BYTES : 0;
}

int64_t gsr_matrix_streamed_bytes(const gsr_matrix* A) { return A ? A->so.h2d_bytes : 0; }

int gsr_matrix_append_rows(gsr_matrix* A, int64_t row0, int64_t nrows, const int32_t* star,
                           const int32_t* att, const int32_t* instr, const double* vals) {
    if (!A) return GSR_EINVAL;
    if (A->state != 0) return GSR_ESTATE;
    if (nrows < 0 || row0 != A->rows_appended || row0 + nrows > A->dims.n_rows) return GSR_EINVAL;
    if (nrows == 0) return GSR_OK;
    if (!star || !att || !instr || !vals) return GSR_EINVAL;
    // host or device arrays: cudaMemcpyDefault resolves the direction per pointer
    for (int64_t r0 = 0; r0 < nrows;) {
        int64_t nr = A->seg_cap - A->seg_fill;
        if (nr > nrows - r0) nr = nrows - r0;
        const int64_t f = A->seg_fill;
        GSR_CUDA_TRY(cudaMemcpyAsync(A->st_star + f, star + r0, (size_t)nr * 4, cudaMemcpyDefault, A->stream));
        GSR_CUDA_TRY(cudaMemcpyAsync(A->st_att + f, att + r0, (size_t)nr * 4, cudaMemcpyDefault, A->stream));
        GSR_CUDA_TRY(cudaMemcpyAsync(A->st_instr + 6 * f, instr + 6 * r0, (size_t)nr * 24, cudaMemcpyDefault, A->stream));
        GSR_CUDA_TRY(cudaMemcpyAsync(A->st_vals + 24 * f, vals + 24 * r0, (size_t)nr * 192, cudaMemcpyDefault, A->stream));
        A->seg_fill += nr;
        A->rows_appended += nr;
        r0 += nr;
        if (A->seg_fill == A->seg_cap || A->rows_appended == A->dims.n_rows) GSR_TRY(flush_segment(A));
    }
    // the caller may free or overwrite its arrays once this returns
    GSR_CUDA_TRY(cudaStreamSynchronize(A->stream));
    return GSR_OK;
}

int gsr_matrix_finalize(gsr_matrix* A) {
    if (!A) return GSR_EINVAL;
    if (A->state != 0) return GSR_ESTATE;
    if (A->rows_appended != A->dims.n_rows) return GSR_ESTATE;
    GSR_TRY(flush_segment(A));
    int err = 0;
    GSR_CUDA_TRY(cudaMemcpyAsync(&err, A->err, sizeof(int), cudaMemcpyDeviceToHost, A->stream));
    GSR_CUDA_TRY(cudaStreamSynchronize(A->stream));
    free_staging(A);
    if (err != 0) return GSR_EINVAL;
    A->n_units = (int)A->units_host->size();
    A->m_int = A->n_tiles * R;
    GSR_TRY(dev_alloc(A, (void**)&A->units, (size_t)(A->n_units > 0 ? A->n_units : 1) * sizeof(Unit)));
    if (A->n_units > 0) {
        GSR_CUDA_TRY(cudaMemcpyAsync(A->units, A->units_host->data(), (size_t)A->n_units * sizeof(Unit),
                                     cudaMemcpyHostToDevice, A->stream));
        if (!A->so.on) GSR_TRY(finish_tiles(A, A->tiles, 0, A->n_tiles));   // (streamed: per segment)
    }
    GSR_CUDA_TRY(cudaStreamSynchronize(A->stream));
    if (A->so.on) {
        // chunk table: the leading units that lie wholly on the device form the resident view,
        // the rest is cut into runs of whole units of at most chunk_cap tiles
        StreamStore& so = A->so;
        dev_free(A, so.seg, (size_t)so.seg_cap * TILE_BYTES);
        so.seg = nullptr;
        const std::vector<Unit>& U = *A->units_host;
        int u = 0;
        while (u < A->n_units && (int64_t)U[u].tile0 + U[u].ntiles <= so.res_cap) ++u;
        so.res_units = u;
        while (u < A->n_units) {
            Chunk ch{u, u, U[u].tile0, U[u].tile0};
            while (u < A->n_units && (int64_t)U[u].tile0 + U[u].ntiles - ch.t0 <= so.chunk_cap) {
                ch.t1 = (int64_t)U[u].tile0 + U[u].ntiles;
                ch.u1 = ++u;
            }
            so.chunks->push_back(ch);
        }
        for (int b = 0; b < 2; ++b) {
            GSR_TRY(dev_alloc(A, (void**)&so.buf[b], (size_t)so.chunk_cap * TILE_BYTES));
            GSR_CUDA_TRY(cudaEventCreateWithFlags(&so.copied[b], cudaEventDisableTiming));
            GSR_CUDA_TRY(cudaEventCreateWithFlags(&so.done[b], cudaEventDisableTiming));
        }
        GSR_CUDA_TRY(cudaEventCreateWithFlags(&so.fork, cudaEventDisableTiming));
        GSR_CUDA_TRY(cudaStreamCreateWithFlags(&so.copy, cudaStreamNonBlocking));
    }
    GSR_TRY(configure_product_kernels(A));
    A->m_global = A->dims.n_rows;
    A->n_global = A->n_cols;
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
    free_staging(A);
    free_constraints(A);
    free_stream_store(A);
    cudaFree(A->tiles);
    cudaFree(A->perm);
    cudaFree(A->units);
    cudaFree(A->unit_counter);
    cudaFree(A->seg_bin_rows);
    cudaFree(A->last_star);
    cudaFree(A->p);
    cudaFree(A->yint);
    cudaFree(A->err);
    cudaFree(A->coef_one);
    cudaGetLastError();
    delete A->units_host;
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
        case GSR_OPT_FUSED: A->opt_two_pass = value == 0; return GSR_OK;
        case GSR_OPT_FIXED_POINT: A->opt_no_fixed = value == 0; return GSR_OK;
        case GSR_OPT_APROD2_SPLIT:
            if (value < -1 || value > 1) return GSR_EINVAL;
            A->opt_aprod2_split = (int)value + 1;
            return GSR_OK;
        case GSR_OPT_WHILE_GRAPH: A->opt_while = value != 0; return GSR_OK;
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
    auto expand = [&](const TileView& v) -> int {
        const int64_t r0 = v.t0 * R, r1 = v.t1 * R;
        if (r1 <= r0) return GSR_OK;
        k_expand_rows<<<(unsigned)((r1 - r0 + 255) / 256), 256, 0, A->stream>>>(
            v.base, A->perm, r0, r1, row0, nrows, A->dims.n_stars, A->dims.n_dfa, A->dims.n_instr, dc, dv);
        count_launch();
        GSR_CUDA_TRY(cudaGetLastError());
        return GSR_OK;
    };
    int rcv = A->so.on ? for_each_view(const_cast<gsr_matrix*>(A), A->stream, expand)
                       : expand(TileView{A->tiles, 0, A->n_units, 0, A->n_tiles});
    e = rcv == GSR_OK ? cudaGetLastError() : cudaErrorUnknown;
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
    GSR_TRY(launch_con_colsumsq(A, A->p, s));
    if (A->comm)   // column norms of the replicated slice are sums over all row shards
        GSR_TRY(comm_allreduce_sum(A->comm, A->p + A->off_att, (size_t)(A->n_cols - A->off_att), s));
    k_make_p<<<(unsigned)((A->n_cols + 255) / 256), 256, 0, s>>>(A->p, A->n_cols);
    count_launch();
    if (A->n_tiles > 0) {
        auto scale = [&](const TileView& v) -> int {
            const int64_t nt = v.t1 - v.t0;
            if (nt <= 0) return GSR_OK;
            k_scale_values<<<(unsigned)((nt + 7) / 8), 256, 0, s>>>(
                v.base, v.t0, nt, A->p, A->dims.n_stars, A->dims.n_dfa, A->dims.n_instr);
            count_launch();
            GSR_CUDA_TRY(cudaGetLastError());
            return GSR_OK;
        };
        if (A->so.on) GSR_TRY(for_each_view(A, s, scale, /*writeback=*/true));
        else GSR_TRY(scale(TileView{A->tiles, 0, A->n_units, 0, A->n_tiles}));
    }
    GSR_TRY(launch_con_scale(A, A->p, s));
    GSR_CUDA_TRY(cudaGetLastError());
    if (p_out) {
        GSR_CUDA_TRY(cudaMemcpyAsync(p_out, A->p, (size_t)A->n_cols * 8, cudaMemcpyDefault, s));
        if (!is_device_ptr(p_out)) GSR_CUDA_TRY(cudaStreamSynchronize(s));
    }
    return GSR_OK;
}

}  // extern "C"
