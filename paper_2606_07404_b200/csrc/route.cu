// Router: fp32 logits in the canonical order (R1) + warp-level top-k + softmax over the selected.
// PAPER.md L224 (routing logits + per-expert bias), L239 (top-k over real experts); BASELINE.json configs[0]
// (softmax over the selected logits, ties -> lower expert id).
#include "common.cuh"

namespace tqp {

// logits[t][e] = fmaf-chain over i ascending (bit-exact against the oracle: one accumulator per (t,e),
// no split-K).  Register-tiled fp32 "SGEMM" on the FMA pipes: block = 128 tokens x 64 experts, 256 threads,
// each thread 8 tokens x 4 experts.  X is bf16 (widened exactly), W_r fp32.
constexpr int RT_TOK = 128, RT_EXP = 64, RT_K = 32;

__global__ void __launch_bounds__(256) route_logits_kernel(const bf16 *__restrict__ X, const float *__restrict__ W_r,
                                                           const float *__restrict__ bias, float *__restrict__ logits,
                                                           int T, int d, int E) {
    __shared__ float xs[RT_K][RT_TOK + 4];   // [i][token]
    __shared__ float wsm[RT_K][RT_EXP];      // [i][expert]
    const int tid = threadIdx.x;
    const int t0 = blockIdx.x * RT_TOK, e0 = blockIdx.y * RT_EXP;
    const int tx = tid % 16, ty = tid / 16;  // tx -> experts (4 each), ty -> tokens (8 each)
    float acc[8][4];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.f;

    for (int i0 = 0; i0 < d; i0 += RT_K) {
        // X tile: 128 tokens x 32 i (bf16).  Each thread loads 16 contiguous bytes (8 values) x 2.
        for (int v = tid; v < RT_TOK * RT_K / 8; v += 256) {
            int tok = v / (RT_K / 8), seg = v % (RT_K / 8);
            uint4 raw = make_uint4(0, 0, 0, 0);
            if (t0 + tok < T) raw = *reinterpret_cast<const uint4 *>(X + (size_t)(t0 + tok) * d + i0 + seg * 8);
            const uint32_t *r = reinterpret_cast<const uint32_t *>(&raw);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                float2 f = bf16x2_to_float2(r[q]);
                xs[seg * 8 + 2 * q][tok] = f.x;
                xs[seg * 8 + 2 * q + 1][tok] = f.y;
            }
        }
        for (int v = tid; v < RT_K * RT_EXP; v += 256) {
            int i = v / RT_EXP, e = v % RT_EXP;
            wsm[i][e] = (e0 + e < E) ? W_r[(size_t)(i0 + i) * E + e0 + e] : 0.f;
        }
        __syncthreads();
#pragma unroll 8
        for (int i = 0; i < RT_K; ++i) {
            float xv[8], wv[4];
            float4 x0 = *reinterpret_cast<const float4 *>(&xs[i][ty * 8]);
            float4 x1 = *reinterpret_cast<const float4 *>(&xs[i][ty * 8 + 4]);
            xv[0] = x0.x; xv[1] = x0.y; xv[2] = x0.z; xv[3] = x0.w;
            xv[4] = x1.x; xv[5] = x1.y; xv[6] = x1.z; xv[7] = x1.w;
            float4 w0 = *reinterpret_cast<const float4 *>(&wsm[i][tx * 4]);
            wv[0] = w0.x; wv[1] = w0.y; wv[2] = w0.z; wv[3] = w0.w;
#pragma unroll
            for (int a = 0; a < 8; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) acc[a][b] = fmaf(xv[a], wv[b], acc[a][b]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        int t = t0 + ty * 8 + a;
        if (t >= T) continue;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            int e = e0 + tx * 4 + b;
            if (e < E) {
                float v = acc[a][b];
                if (bias) v = v + bias[e];
                logits[(size_t)t * E + e] = v;
            }
        }
    }
}

// One warp per token: k rounds of a warp arg-max under the total order (-logit, id); then the softmax over
// the k selected logits with the sum taken in ascending j (the oracle's order).  E <= 1024.
__global__ void __launch_bounds__(128) route_topk_kernel(const float *__restrict__ logits, int32_t *__restrict__ topk_idx,
                                                         float *__restrict__ topk_w, int T, int E, int k) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (warp >= T) return;
    const float *l = logits + (size_t)warp * E;
    constexpr int PER = 32;  // E <= 1024
    float v[PER];
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        int e = q * 32 + lane;
        v[q] = (e < E) ? l[e] : -INFINITY;
    }
    uint32_t taken = 0;  // bit q: slot q of this lane already selected
    float sel_l = 0.f;   // lane j keeps the j-th selected logit
    int sel_e = 0;
    for (int j = 0; j < k; ++j) {
        float bv = -INFINITY;
        int be = 0x7fffffff;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            int e = q * 32 + lane;
            bool ok = (e < E) && !((taken >> q) & 1u);
            if (ok && (v[q] > bv || be == 0x7fffffff)) { bv = v[q]; be = e; }   // ascending e: ties keep lower id
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            float ov = __shfl_xor_sync(0xffffffffu, bv, off);
            int oe = __shfl_xor_sync(0xffffffffu, be, off);
            bool better = (oe != 0x7fffffff) && (be == 0x7fffffff || ov > bv || (ov == bv && oe < be));
            if (better) { bv = ov; be = oe; }
        }
        if ((be % 32) == lane) taken |= 1u << (be / 32);
        if (lane == j) { sel_l = bv; sel_e = be; }
    }
    float m = __shfl_sync(0xffffffffu, sel_l, 0);
    float ex = (lane < k) ? expf(sel_l - m) : 0.f;
    float sum = 0.f;
    for (int j = 0; j < k; ++j) sum = sum + __shfl_sync(0xffffffffu, ex, j);
    if (lane < k) {
        topk_idx[(size_t)warp * k + lane] = sel_e;
        topk_w[(size_t)warp * k + lane] = ex / sum;
    }
}

tqp_status launch_route(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *bias, int32_t *topk_idx,
                        float *topk_w, float *logits, cudaStream_t s) {
    const int d = c->desc.d, E = c->desc.E, k = c->desc.k;
    dim3 grid((T + RT_TOK - 1) / RT_TOK, (E + RT_EXP - 1) / RT_EXP);
    route_logits_kernel<<<grid, 256, 0, s>>>(X, W_r, bias, logits, T, d, E);
    TQP_LAUNCH_OK(c);
    route_topk_kernel<<<(T + 3) / 4, 128, 0, s>>>(logits, topk_idx, topk_w, T, E, k);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
