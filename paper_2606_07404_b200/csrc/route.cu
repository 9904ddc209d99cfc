// Router: fp32 logits in the canonical order (R1) + warp-level top-k + softmax over the selected.
// PAPER.md L224 (routing logits + per-expert bias), L239 (top-k over real experts); BASELINE.json configs[0]
// (softmax over the selected logits, ties -> lower expert id).
#include "common.cuh"

namespace tqp {

// logits[t][e] = fmaf-chain over i ascending (bit-exact against the oracle: one accumulator per (t,e),
// no split-K).  Register-tiled fp32 "SGEMM" on the FMA pipes: block = 64 tokens x 96 experts, 128 threads,
// each thread 8 tokens x 6 experts (48 FMAs per 5 shared-memory loads), K-chunks of 32 double-buffered in shared
// memory (W_r by cp.async, X through registers: bf16 widened exactly and stored transposed).  Bound: fp32 FMA
// issue rate (R1 forbids tensor cores and any re-association of the sum).
constexpr int RT_TOK = 64, RT_EXP = 96, RT_K = 32, RT_XLD = RT_TOK + 4;

__global__ void __launch_bounds__(128) route_logits_kernel(const bf16 *__restrict__ X, const float *__restrict__ W_r,
                                                           const float *__restrict__ bias, float *__restrict__ logits,
                                                           int T, int d, int E) {
    __shared__ __align__(16) float xs[2][RT_K][RT_XLD];   // [buf][i][token]
    __shared__ __align__(16) float wsm[2][RT_K][RT_EXP];  // [buf][i][expert]
    const int tid = threadIdx.x;
    const int t0 = blockIdx.x * RT_TOK, e0 = blockIdx.y * RT_EXP;
    const int tx = tid % 16, ty = tid / 16;   // tx -> experts (6 each), ty -> tokens (8 each)
    const bool w_vec = (E % 4) == 0;          // 16-byte cp.async needs aligned rows and whole chunks
    float acc[8][6];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 6; ++b) acc[a][b] = 0.f;

    // X tile: 64 tokens x 32 i (bf16) = 256 chunks of 8 values; thread owns chunks (token = tid % 64, seg = tid / 64 + 2 j)
    const int xtok = tid % RT_TOK, xseg = tid / RT_TOK;
    const bool x_ok = t0 + xtok < T;
    const bf16 *xsrc = X + (size_t)(x_ok ? t0 + xtok : 0) * d + xseg * 8;
    uint4 xr[2];
    auto load_x = [&](int i0) {
#pragma unroll
        for (int j = 0; j < 2; ++j)
            xr[j] = x_ok ? *reinterpret_cast<const uint4 *>(xsrc + i0 + j * 16) : make_uint4(0, 0, 0, 0);
    };
    auto store_x = [&](int buf) {
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const uint32_t *r = reinterpret_cast<const uint32_t *>(&xr[j]);
            const int ib = (xseg + 2 * j) * 8;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                float2 f = bf16x2_to_float2(r[q]);
                xs[buf][ib + 2 * q][xtok] = f.x;
                xs[buf][ib + 2 * q + 1][xtok] = f.y;
            }
        }
    };
    auto load_w = [&](int i0, int buf) {
        if (w_vec) {
            for (int v = tid; v < RT_K * RT_EXP / 4; v += 128) {
                const int i = v / (RT_EXP / 4), e = (v % (RT_EXP / 4)) * 4;
                const bool ok = e0 + e < E;
                const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&wsm[buf][i][e]);
                const float *src = W_r + (size_t)(i0 + i) * E + (ok ? e0 + e : 0);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(ok ? 16 : 0) : "memory");
            }
        } else {
            for (int v = tid; v < RT_K * RT_EXP; v += 128) {
                const int i = v / RT_EXP, e = v % RT_EXP;
                wsm[buf][i][e] = (e0 + e < E) ? W_r[(size_t)(i0 + i) * E + e0 + e] : 0.f;
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    load_x(0);
    load_w(0, 0);
    store_x(0);
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    const int nc = d / RT_K;
    for (int c = 0; c < nc; ++c) {
        const int buf = c & 1;
        if (c + 1 < nc) {
            load_x((c + 1) * RT_K);
            load_w((c + 1) * RT_K, buf ^ 1);
        }
#pragma unroll 8
        for (int i = 0; i < RT_K; ++i) {
            const float4 x0 = *reinterpret_cast<const float4 *>(&xs[buf][i][ty * 8]);
            const float4 x1 = *reinterpret_cast<const float4 *>(&xs[buf][i][ty * 8 + 4]);
            const float2 w0 = *reinterpret_cast<const float2 *>(&wsm[buf][i][tx * 6]);
            const float2 w1 = *reinterpret_cast<const float2 *>(&wsm[buf][i][tx * 6 + 2]);
            const float2 w2 = *reinterpret_cast<const float2 *>(&wsm[buf][i][tx * 6 + 4]);
            const float xv[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
            const float wv[6] = {w0.x, w0.y, w1.x, w1.y, w2.x, w2.y};
#pragma unroll
            for (int a = 0; a < 8; ++a)
#pragma unroll
                for (int b = 0; b < 6; ++b) acc[a][b] = fmaf(xv[a], wv[b], acc[a][b]);
        }
        if (c + 1 < nc) {
            store_x(buf ^ 1);
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        const int t = t0 + ty * 8 + a;
        if (t >= T) continue;
#pragma unroll
        for (int b = 0; b < 6; ++b) {
            const int e = e0 + tx * 6 + b;
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
    route_logits_kernel<<<grid, 128, 0, s>>>(X, W_r, bias, logits, T, d, E);
    TQP_LAUNCH_OK(c);
    route_topk_kernel<<<(T + 3) / 4, 128, 0, s>>>(logits, topk_idx, topk_w, T, E, k);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
