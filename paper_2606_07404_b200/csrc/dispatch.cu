// Dispatch: stable counting sort of the flat assignments a = t*k+j by expert id (histogram / scan / ranked
// scatter), bit-exact against the oracle, plus the device-side tile list of the grouped GEMMs.
// PAPER.md L289 ("MoE routing and expert dispatch"), L553 ("grouped MoE expert computation").
#include "common.cuh"

namespace tqp {

// Phase 1: each warp owns one chunk of kDispChunk consecutive assignments and counts them per expert.
__global__ void __launch_bounds__(128) dispatch_hist_kernel(const int32_t *__restrict__ topk_idx, int N, int E,
                                                            int32_t *__restrict__ blk_counts) {
    extern __shared__ int32_t sm[];
    const int warp_in_blk = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int chunk = blockIdx.x * 4 + warp_in_blk;
    int32_t *cnt = sm + warp_in_blk * E;
    for (int e = lane; e < E; e += 32) cnt[e] = 0;
    __syncwarp();
    const int a0 = chunk * kDispChunk;
    for (int i = lane; i < kDispChunk; i += 32) {
        int a = a0 + i;
        if (a < N) atomicAdd(&cnt[topk_idx[a]], 1);
    }
    __syncwarp();
    if (a0 < N)
        for (int e = lane; e < E; e += 32) blk_counts[(size_t)chunk * E + e] = cnt[e];
}

// Phase 2a: one warp per expert turns its column of chunk counts into exclusive prefixes (in place) and writes the
// expert's total.  Phase 2b (one block): exclusive scan over experts -> offsets, and the GEMM tile list.
__global__ void __launch_bounds__(256) dispatch_scan_chunks_kernel(int32_t *__restrict__ blk_counts, int nchunks, int E,
                                                                   int32_t *__restrict__ counts) {
    const int e = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (e >= E) return;
    int running = 0;
    for (int c0 = 0; c0 < nchunks; c0 += 32) {
        const int c = c0 + lane;
        const int v = (c < nchunks) ? blk_counts[(size_t)c * E + e] : 0;
        int incl = v;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t;
        }
        if (c < nchunks) blk_counts[(size_t)c * E + e] = running + incl - v;
        running += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) counts[e] = running;
}

__global__ void __launch_bounds__(1024) dispatch_scan_experts_kernel(const int32_t *__restrict__ counts, int E,
                                                                     int32_t *__restrict__ offsets, Tile *__restrict__ tiles,
                                                                     int32_t *__restrict__ num_tiles, int tile_rows,
                                                                     Tile *__restrict__ xsegs, int32_t *__restrict__ xfirst,
                                                                     int32_t *__restrict__ tfirst) {
    __shared__ int32_t w_off[32], w_til[32], w_xs[32];
    const int e = threadIdx.x, lane = e % 32, warp = e / 32;
    const int cnt = (e < E) ? counts[e] : 0;
    const int nt = (cnt + tile_rows - 1) / tile_rows;
    const int nx = max(0, (cnt + kWgradSeg - 1) / kWgradSeg - 1);   // row segments of this expert beyond its first (weight gradients)
    int io = cnt, it = nt, ix = nx;   // inclusive scans inside the warp
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        int a = __shfl_up_sync(0xffffffffu, io, off), b = __shfl_up_sync(0xffffffffu, it, off);
        int c = __shfl_up_sync(0xffffffffu, ix, off);
        if (lane >= off) { io += a; it += b; ix += c; }
    }
    if (lane == 31) { w_off[warp] = io; w_til[warp] = it; w_xs[warp] = ix; }
    __syncthreads();
    if (warp == 0) {
        int a = w_off[lane], b = w_til[lane], c = w_xs[lane], ia = a, ib = b, ic = c;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            int x = __shfl_up_sync(0xffffffffu, ia, off), y = __shfl_up_sync(0xffffffffu, ib, off);
            int z = __shfl_up_sync(0xffffffffu, ic, off);
            if (lane >= off) { ia += x; ib += y; ic += z; }
        }
        w_off[lane] = ia - a;   // exclusive prefix of the warp totals
        w_til[lane] = ib - b;
        w_xs[lane] = ic - c;
    }
    __syncthreads();
    const int off_e = w_off[warp] + io - cnt, til_e = w_til[warp] + it - nt, xs_e = w_xs[warp] + ix - nx;
    if (e < E) {
        // extra row segments of experts with more than kWgradSeg rows: segment i+1 covers rows [(i+1) S, (i+2) S) of the expert
        xfirst[e] = xs_e;
        if (e == E - 1) xfirst[E] = xs_e + nx;
        for (int i = 0; i < nx; ++i) {
            Tile t;
            t.expert = e;
            t.row0 = off_e + (i + 1) * kWgradSeg;
            t.rows = min(kWgradSeg, cnt - (i + 1) * kWgradSeg);
            t.pad = i + 1;
            xsegs[xs_e + i] = t;
        }
        offsets[e] = off_e;
        tfirst[e] = til_e;   // the expert's tiles are [tfirst[e], tfirst[e + 1])
        if (e == E - 1) { offsets[E] = off_e + cnt; *num_tiles = til_e + nt; tfirst[E] = til_e + nt; }
        if (nt > 0) {
            int per = (cnt + nt - 1) / nt;
            per = (per + 15) & ~15;   // balanced tiles, multiples of 16 rows (UMMA N granularity)
            for (int i = 0; i < nt; ++i) {
                Tile t;
                t.expert = e;
                t.row0 = off_e + i * per;
                t.rows = max(0, min(per, cnt - i * per));   // rows == 0: skipped by the consumers
                t.pad = 0;
                tiles[til_e + i] = t;
            }
        }
    }
}

// Phase 3: ranked scatter.  Inside a chunk the 32-wide groups are processed in order; __match_any_sync gives
// the rank among equal experts inside a group, so rows of one expert stay in ascending a (stable).
__global__ void __launch_bounds__(128) dispatch_scatter_kernel(const int32_t *__restrict__ topk_idx, int N, int E,
                                                               const int32_t *__restrict__ blk_base,
                                                               const int32_t *__restrict__ offsets,
                                                               int32_t *__restrict__ perm, int32_t *__restrict__ inv_perm) {
    extern __shared__ int32_t sm[];
    const int warp_in_blk = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int chunk = blockIdx.x * 4 + warp_in_blk;
    const int a0 = chunk * kDispChunk;
    if (a0 >= N) return;
    int32_t *cur = sm + warp_in_blk * E;
    for (int e = lane; e < E; e += 32) cur[e] = blk_base[(size_t)chunk * E + e] + offsets[e];
    __syncwarp();
    for (int i = 0; i < kDispChunk; i += 32) {
        int a = a0 + i + lane;
        bool valid = a < N;
        int e = valid ? topk_idx[a] : -1 - lane;   // invalid lanes get unique keys
        uint32_t peers = __match_any_sync(0xffffffffu, e);
        int rank = __popc(peers & ((1u << lane) - 1u));
        int p = 0;
        if (valid) p = cur[e] + rank;
        __syncwarp();
        if (valid && rank == 0) cur[e] += __popc(peers);   // one leader per expert in this group
        __syncwarp();
        if (valid) {
            perm[p] = a;
            inv_perm[a] = p;
        }
    }
}

tqp_status launch_dispatch(tqp_ctx *c, int T, const int32_t *topk_idx, int32_t *counts, int32_t *offsets,
                           int32_t *perm, int32_t *inv_perm, cudaStream_t s) {
    const int E = c->desc.E, N = T * c->desc.k;
    const int nchunks = (N + kDispChunk - 1) / kDispChunk;
    const int nblk = (nchunks + 3) / 4;
    int32_t *blk = c->p<int32_t>(c->ws.blk_counts);
    const size_t smem = (size_t)4 * E * sizeof(int32_t);
    dispatch_hist_kernel<<<nblk, 128, smem, s>>>(topk_idx, N, E, blk);
    TQP_LAUNCH_OK(c);
    dispatch_scan_chunks_kernel<<<(E + 7) / 8, 256, 0, s>>>(blk, nchunks, E, counts);
    TQP_LAUNCH_OK(c);
    dispatch_scan_experts_kernel<<<1, 1024, 0, s>>>(counts, E, offsets, c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles), kTileRows,
                                                    c->p<Tile>(c->ws.xsegs), c->p<int32_t>(c->ws.xfirst), c->p<int32_t>(c->ws.tfirst));
    TQP_LAUNCH_OK(c);
    dispatch_scatter_kernel<<<nblk, 128, smem, s>>>(topk_idx, N, E, blk, offsets, perm, inv_perm);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
