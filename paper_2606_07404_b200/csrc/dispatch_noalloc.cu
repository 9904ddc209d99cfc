// tqp_dispatch_noalloc: the dispatch of dispatch.cu (stable counting sort of a = t*k+j by expert id; "expert
// dispatch") for callers that cannot allocate -- no ctx, no workspace, no cudaMalloc / cudaFree or any allocating call.
// Its only scratch, the per-chunk histograms, lives in a file-scope __device__ array of fixed size.
//
// The three kernels are this file's own variants of dispatch_hist / dispatch_scan_chunks / dispatch_scatter (same
// algorithm, hence the same bits: counts, offsets, perm and inv_perm equal tqp_dispatch's); the expert scan writes
// offsets only (the grouped-GEMM tile list belongs to a ctx and is not built here).
//
// Sharing.  Every call on a device uses the SAME array.  Nothing in it has to start at zero: phase 1 overwrites every entry
// the later phases read (chunks [0, nchunks) x experts [0, E)), so the previous call's contents are never seen.  Two calls
// that overlap on the GPU (different streams, or a graph replayed beside a live call) race on it and give garbage; calls on
// one stream are ordered and safe.  Each GPU that loads the library holds the 4 MiB until the process exits.
#include <cstdio>
#include <mutex>

#include "common.cuh"

namespace {

constexpr int kNoAllocChunk = tqp::kDispChunk;              // assignments per warp, as in dispatch.cu
constexpr size_t kNoAllocScratchInts = (size_t)1 << 20;     // 4 MiB: ceil(T k / 256) * E <= 1 048 576
constexpr int kMaxDevices = 64;

static __device__ __align__(256) int32_t g_dispatch_scratch[kNoAllocScratchInts];   // [nchunks][E] chunk histograms / bases

thread_local char t_err[256] = "";

// Phase 1: each warp owns one chunk of consecutive assignments and counts them per expert (always writes its E entries).
__global__ void __launch_bounds__(128) na_hist_kernel(const int32_t *__restrict__ topk_idx, int N, int E, int32_t *__restrict__ blk) {
    extern __shared__ int32_t sm[];
    const int wib = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int chunk = blockIdx.x * 4 + wib, a0 = chunk * kNoAllocChunk;
    if (a0 >= N) return;
    int32_t *cnt = sm + wib * E;
    for (int e = lane; e < E; e += 32) cnt[e] = 0;
    __syncwarp();
    for (int i = lane; i < kNoAllocChunk; i += 32)
        if (a0 + i < N) atomicAdd(&cnt[topk_idx[a0 + i]], 1);
    __syncwarp();
    for (int e = lane; e < E; e += 32) blk[(size_t)chunk * E + e] = cnt[e];
}

// Phase 2a: one warp per expert: its column of chunk counts -> exclusive prefixes (in place), and the expert's total.
__global__ void __launch_bounds__(256) na_scan_chunks_kernel(int32_t *__restrict__ blk, int nchunks, int E, int32_t *__restrict__ counts) {
    const int e = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (e >= E) return;
    int running = 0;
    for (int c0 = 0; c0 < nchunks; c0 += 32) {
        const int c = c0 + lane;
        const int v = (c < nchunks) ? blk[(size_t)c * E + e] : 0;
        int incl = v;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t;
        }
        if (c < nchunks) blk[(size_t)c * E + e] = running + incl - v;
        running += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) counts[e] = running;
}

// Phase 2b (one block of 1024 threads, E <= 1024): exclusive scan of the counts -> offsets[0 .. E].
__global__ void __launch_bounds__(1024) na_scan_experts_kernel(const int32_t *__restrict__ counts, int E, int32_t *__restrict__ offsets) {
    __shared__ int32_t w_off[32];
    const int e = threadIdx.x, lane = e % 32, warp = e / 32;
    const int cnt = (e < E) ? counts[e] : 0;
    int io = cnt;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const int a = __shfl_up_sync(0xffffffffu, io, off);
        if (lane >= off) io += a;
    }
    if (lane == 31) w_off[warp] = io;
    __syncthreads();
    if (warp == 0) {
        const int a = w_off[lane];
        int ia = a;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int x = __shfl_up_sync(0xffffffffu, ia, off);
            if (lane >= off) ia += x;
        }
        w_off[lane] = ia - a;
    }
    __syncthreads();
    if (e < E) {
        const int off_e = w_off[warp] + io - cnt;
        offsets[e] = off_e;
        if (e == E - 1) offsets[E] = off_e + cnt;
    }
}

// Phase 3: ranked scatter; __match_any_sync ranks equal experts inside a 32-wide group, groups run in order (stable).
__global__ void __launch_bounds__(128) na_scatter_kernel(const int32_t *__restrict__ topk_idx, int N, int E, const int32_t *__restrict__ blk,
                                                         const int32_t *__restrict__ offsets, int32_t *__restrict__ perm,
                                                         int32_t *__restrict__ inv_perm) {
    extern __shared__ int32_t sm[];
    const int wib = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int chunk = blockIdx.x * 4 + wib, a0 = chunk * kNoAllocChunk;
    if (a0 >= N) return;
    int32_t *cur = sm + wib * E;
    for (int e = lane; e < E; e += 32) cur[e] = blk[(size_t)chunk * E + e] + offsets[e];
    __syncwarp();
    for (int i = 0; i < kNoAllocChunk; i += 32) {
        const int a = a0 + i + lane;
        const bool valid = a < N;
        const int e = valid ? topk_idx[a] : -1 - lane;   // invalid lanes get unique keys
        const uint32_t peers = __match_any_sync(0xffffffffu, e);
        const int rank = __popc(peers & ((1u << lane) - 1u));
        int p = 0;
        if (valid) p = cur[e] + rank;
        __syncwarp();
        if (valid && rank == 0) cur[e] += __popc(peers);
        __syncwarp();
        if (valid) {
            perm[p] = a;
            inv_perm[a] = p;
        }
    }
}

// Device address of the scratch array, looked up once per device with that device current.  In host code the array's NAME is
// only a host-side stand-in for the symbol: the kernels must be given the address cudaGetSymbolAddress returns.
int32_t *scratch_of_current_device(int *dev_out) {
    static std::mutex mu;
    static int32_t *ptrs[kMaxDevices] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        snprintf(t_err, sizeof t_err, "tqp_dispatch_noalloc: cudaGetDevice: %s (device %d)", cudaGetErrorString(e), dev);
        return nullptr;
    }
    *dev_out = dev;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_dispatch_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(t_err, sizeof t_err, "tqp_dispatch_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return nullptr;
        }
        ptrs[dev] = static_cast<int32_t *>(p);
    }
    return ptrs[dev];
}

}  // namespace

extern "C" {

size_t tqp_dispatch_noalloc_capacity(void) { return kNoAllocScratchInts; }

const char *tqp_dispatch_noalloc_error(void) { return t_err; }

tqp_status tqp_dispatch_noalloc(int T, int k, int E, const int32_t *topk_idx, int32_t *counts, int32_t *offsets, int32_t *perm,
                                int32_t *inv_perm, void *stream) {
    t_err[0] = 0;
    if (!topk_idx || !counts || !offsets || !perm || !inv_perm) {
        snprintf(t_err, sizeof t_err, "tqp_dispatch_noalloc: NULL pointer");
        return TQP_ERR_ARG;
    }
    if (T <= 0 || k <= 0 || k > 32 || E <= 0 || E > 1024 || k > E || (long long)T * k >= (1ll << 31) / 64) {
        snprintf(t_err, sizeof t_err, "tqp_dispatch_noalloc: need T > 0, 1 <= k <= min(32, E), 1 <= E <= 1024, T k < 2^25 (got T=%d k=%d E=%d)", T, k, E);
        return TQP_ERR_ARG;
    }
    const int N = T * k, nchunks = (N + kNoAllocChunk - 1) / kNoAllocChunk;
    if ((size_t)nchunks * (size_t)E > kNoAllocScratchInts) {
        snprintf(t_err, sizeof t_err,
                 "tqp_dispatch_noalloc: ceil(T k / %d) * E = %zu exceeds the static scratch of %zu entries (4 MiB); use tqp_dispatch with a workspace",
                 kNoAllocChunk, (size_t)nchunks * (size_t)E, kNoAllocScratchInts);
        return TQP_ERR_SHAPE;
    }
    int dev = -1;
    int32_t *blk = scratch_of_current_device(&dev);
    if (!blk) return TQP_ERR_CUDA;
    cudaStream_t s = (cudaStream_t)stream;
    const int nblk = (nchunks + 3) / 4;
    const size_t smem = (size_t)4 * E * sizeof(int32_t);   // <= 16 KB: no attribute needed
    na_hist_kernel<<<nblk, 128, smem, s>>>(topk_idx, N, E, blk);
    na_scan_chunks_kernel<<<(E + 7) / 8, 256, 0, s>>>(blk, nchunks, E, counts);
    na_scan_experts_kernel<<<1, 1024, 0, s>>>(counts, E, offsets);
    na_scatter_kernel<<<nblk, 128, smem, s>>>(topk_idx, N, E, blk, offsets, perm, inv_perm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(t_err, sizeof t_err, "tqp_dispatch_noalloc: launch failed: %s", cudaGetErrorString(e));
        return TQP_ERR_CUDA;
    }
    return TQP_OK;
}

}  // extern "C"
