// Router: fp32 logits in the canonical order (R1) + warp-level top-k + softmax over the selected.
// PAPER.md L224 (routing logits + per-expert bias), L239 (top-k over real experts); BASELINE.json configs[0]
// (softmax over the selected logits, ties -> lower expert id).
#include "common.cuh"

namespace tqp {

// logits[t][e] = fmaf-chain over i ascending (bit-exact against the oracle: one accumulator per (t,e),
// no split-K).  Register-tiled fp32 "SGEMM" on the FMA pipes: block = 96 tokens x 96 experts, 128 threads,
// each thread 12 tokens x 6 experts (72 FMAs per 6 shared-memory loads), K-chunks of 32 double-buffered in shared
// memory (W_r by cp.async, X through registers: bf16 widened exactly and stored transposed).  96-token tiles make
// 430 CTAs at T = 8192, E = 460: one wave of 3 CTAs per SM on 148 SMs with 97 % of the slots filled (64-token tiles
// gave 640 CTAs on 740 slots: 4 or 5 per SM, 86 %).  Bound: fp32 FMA issue rate (R1 forbids tensor cores and any
// re-association of the sum).
// A second instantiation (4 x 4 per thread: 32 tokens x 64 experts per CTA) serves small problems, where the large tile
// would leave most SMs idle (configs[1]: T = 4096, E = 64 -> 43 large CTAs on 148 SMs, 148 us; 128 small CTAs: see DESIGN).
constexpr int RT_K = 32;

// d.x = fma(a.x, b, d.x), d.y = fma(a.y, b, d.y): two IEEE fp32 FMAs in one instruction (FFMA2 on sm_100: packed
// register pairs with a scalar third operand).  Each lane rounds exactly like fmaf, so the logits stay bit-identical to the
// canonical chain; what changes is the number of instructions per FMA, which is what bounds this kernel.
__device__ __forceinline__ void ffma2(float2 &d, const float2 a, const float b) {
    uint64_t dd, aa, bb;
    asm("mov.b64 %0, {%1,%2};" : "=l"(dd) : "f"(d.x), "f"(d.y));
    asm("mov.b64 %0, {%1,%2};" : "=l"(aa) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1,%1};" : "=l"(bb) : "f"(b));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(dd) : "l"(aa), "l"(bb));
    asm("mov.b64 {%0,%1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(dd));
}

template <int RT_TM, int RT_EN>   // per-thread tile: RT_TM tokens x RT_EN experts; 8 x 16 threads per CTA
__global__ void __launch_bounds__(128, 3) route_logits_kernel(const bf16 *__restrict__ X, const float *__restrict__ W_r,
                                                              const float *__restrict__ bias, float *__restrict__ logits,
                                                              int T, int d, int E) {
    constexpr int RT_TOK = 8 * RT_TM, RT_EXP = 16 * RT_EN, RT_XLD = RT_TOK;   // unpadded rows: transposed stores and broadcast loads are conflict-free
    constexpr int RT_XCH = (RT_TOK * RT_K / 8 + 127) / 128;    // 16-byte X chunks per thread per K-chunk
    constexpr int RT_WCH = RT_K * RT_EXP / 4 / 128;            // 16-byte W_r chunks per thread per K-chunk
    __shared__ __align__(16) float xs[2][RT_K][RT_XLD];   // [buf][i][token]
    __shared__ __align__(16) float wsm[2][RT_K][RT_EXP];  // [buf][i][expert]
    const int tid = threadIdx.x;
    const int t0 = blockIdx.x * RT_TOK, e0 = blockIdx.y * RT_EXP;
    const int tx = tid % 16, ty = tid / 16;   // tx -> experts (6 each), ty -> tokens (12 each)
    const bool w_vec = (E % 4) == 0;          // 16-byte cp.async needs aligned rows and whole chunks
    static_assert(RT_TM % 2 == 0, "token pairs");
    float2 acc[RT_TM / 2][RT_EN];   // (token 2a, token 2a + 1) x expert b
#pragma unroll
    for (int a = 0; a < RT_TM / 2; ++a)
#pragma unroll
        for (int b = 0; b < RT_EN; ++b) acc[a][b] = make_float2(0.f, 0.f);

    // X tile: 96 tokens x 32 i (bf16) = 384 chunks of 8 values; chunk v = tid + 128 j: token v % 96, segment v / 96
    const bf16 *xsrc[RT_XCH];
    int xtok[RT_XCH], xseg[RT_XCH];
#pragma unroll
    for (int j = 0; j < RT_XCH; ++j) {
        const int v = tid + 128 * j;
        xtok[j] = v % RT_TOK;
        xseg[j] = v / RT_TOK;   // segments past the K-chunk (small tile: fewer chunks than threads) load nothing
        xsrc[j] = (xseg[j] < RT_K / 8 && t0 + xtok[j] < T) ? X + (size_t)(t0 + xtok[j]) * d + xseg[j] * 8 : nullptr;
    }
    // W_r tile: 32 i x 96 experts (fp32) = 768 chunks of 4 values; chunk v: row v / 24, experts 4 (v % 24) ..
    const float *wsrc[RT_WCH];
    uint32_t wdst[RT_WCH];
#pragma unroll
    for (int j = 0; j < RT_WCH; ++j) {
        const int v = tid + 128 * j, i = v / (RT_EXP / 4), e = (v % (RT_EXP / 4)) * 4;
        wsrc[j] = (e0 + e < E) ? W_r + (size_t)i * E + e0 + e : nullptr;   // past E: zero-filled
        wdst[j] = (uint32_t)__cvta_generic_to_shared(&wsm[0][i][e]);
    }
    uint4 xr[RT_XCH];
    auto load_x = [&](int i0) {
#pragma unroll
        for (int j = 0; j < RT_XCH; ++j)
            xr[j] = xsrc[j] ? *reinterpret_cast<const uint4 *>(xsrc[j] + i0) : make_uint4(0, 0, 0, 0);
    };
    auto store_x = [&](int buf) {
#pragma unroll
        for (int j = 0; j < RT_XCH; ++j) {
            if (xseg[j] >= RT_K / 8) continue;
            const uint32_t *r = reinterpret_cast<const uint32_t *>(&xr[j]);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                float2 f = bf16x2_to_float2(r[q]);
                xs[buf][xseg[j] * 8 + 2 * q][xtok[j]] = f.x;
                xs[buf][xseg[j] * 8 + 2 * q + 1][xtok[j]] = f.y;
            }
        }
    };
    auto load_w = [&](int i0, int buf) {
        if (w_vec) {
#pragma unroll
            for (int j = 0; j < RT_WCH; ++j) {
                const float *src = wsrc[j] ? wsrc[j] + (size_t)i0 * E : W_r;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(wdst[j] + buf * (uint32_t)sizeof(wsm[0])), "l"(src),
                             "r"(wsrc[j] ? 16 : 0) : "memory");
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
#pragma unroll 4
        for (int i = 0; i < RT_K; ++i) {
            float xv[RT_TM], wv[RT_EN];
#pragma unroll
            for (int a = 0; a < RT_TM / 4; ++a) {
                const float4 x4 = *reinterpret_cast<const float4 *>(&xs[buf][i][ty * RT_TM + 4 * a]);
                xv[4 * a] = x4.x; xv[4 * a + 1] = x4.y; xv[4 * a + 2] = x4.z; xv[4 * a + 3] = x4.w;
            }
#pragma unroll
            for (int b = 0; b < RT_EN / 2; ++b) {
                const float2 w2 = *reinterpret_cast<const float2 *>(&wsm[buf][i][tx * RT_EN + 2 * b]);
                wv[2 * b] = w2.x; wv[2 * b + 1] = w2.y;
            }
#pragma unroll
            for (int a = 0; a < RT_TM / 2; ++a)
#pragma unroll
                for (int b = 0; b < RT_EN; ++b) ffma2(acc[a][b], make_float2(xv[2 * a], xv[2 * a + 1]), wv[b]);
        }
        if (c + 1 < nc) {
            store_x(buf ^ 1);
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < RT_TM; ++a) {
        const int t = t0 + ty * RT_TM + a;
        if (t >= T) continue;
#pragma unroll
        for (int b = 0; b < RT_EN; ++b) {
            const int e = e0 + tx * RT_EN + b;
            if (e < E) {
                float v = (a & 1) ? acc[a / 2][b].y : acc[a / 2][b].x;
                if (bias) v = v + bias[e];
                logits[(size_t)t * E + e] = v;
            }
        }
    }
}

// One warp per token: k rounds of a warp arg-max under the total order (-logit, id); then the softmax over
// the k selected logits with the sum taken in ascending j (the oracle's order).  E <= 1024.
//
// The arg-max works on order-preserving 32-bit integer keys of the floats (sign bit flipped for positives, all bits for
// negatives; -0 is first made +0 so that equal floats have equal keys): a lane's best is a max tree over its PER keys,
// the warp's best one redux.sync (max), the tie-break a second redux.sync (min) over the ids of the slots that hold that
// key.  Key 0 (a NaN pattern no logit maps to) marks slots past E and slots already taken.  (The first version compared
// floats through five rounds of shuffles per selection: 35 us at cfg 2, latency-bound.)
__device__ __forceinline__ uint32_t order_key(float f) {
    if (f == 0.f) f = 0.f;   // -0 -> +0
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float key_value(uint32_t key) { return __uint_as_float((key & 0x80000000u) ? (key ^ 0x80000000u) : ~key); }

// Selects the best remaining slot of the warp: returns its expert id, its key in `best`, and retires it.
template <int PER>
__device__ __forceinline__ int warp_select(uint32_t (&key)[PER], int lane, uint32_t &best) {
    uint32_t t[PER];
#pragma unroll
    for (int q = 0; q < PER; ++q) t[q] = key[q];
#pragma unroll
    for (int s = PER / 2; s > 0; s >>= 1)
#pragma unroll
        for (int q = 0; q < s; ++q) t[q] = max(t[q], t[q + s]);
    const uint32_t m = __reduce_max_sync(0xffffffffu, t[0]);
    int cand = 0x7fffffff;
#pragma unroll
    for (int q = PER - 1; q >= 0; --q)
        if (key[q] == m) cand = q * 32 + lane;   // descending q: the lowest id of this lane survives
    const int e = __reduce_min_sync(0xffffffffu, cand);   // ties -> lower expert id
#pragma unroll
    for (int q = 0; q < PER; ++q)
        if (q * 32 + lane == e) key[q] = 0u;
    best = m;
    return e;
}

template <int PER>   // PER = ceil(E / 32) rounded up to a power of two: logits held per lane
__global__ void __launch_bounds__(128) route_topk_kernel(const float *__restrict__ logits, int32_t *__restrict__ topk_idx,
                                                         float *__restrict__ topk_w, int T, int E, int k) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (warp >= T) return;
    const float *l = logits + (size_t)warp * E;
    uint32_t key[PER];
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        const int e = q * 32 + lane;
        key[q] = (e < E) ? order_key(l[e]) : 0u;
    }
    float sel_l = 0.f;   // lane j keeps the j-th selected logit
    int sel_e = 0;
    for (int j = 0; j < k; ++j) {
        uint32_t m;
        const int e = warp_select<PER>(key, lane, m);
        if (lane == j) { sel_l = key_value(m); sel_e = e; }
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

// Paper-faithful variant: selection by logit + bias, gate values from the sigmoid of the UNBIASED logit,
// normalised over the selected set.  Same warp arg-max as above on the biased keys.
template <int PER>
__global__ void __launch_bounds__(128) route_topk_sigmoid_kernel(const float *__restrict__ logits, const float *__restrict__ bias,
                                                                 int32_t *__restrict__ topk_idx, float *__restrict__ topk_w,
                                                                 float *__restrict__ topk_s, int T, int E, int k) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (warp >= T) return;
    const float *l = logits + (size_t)warp * E;
    uint32_t key[PER];
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        const int e = q * 32 + lane;
        key[q] = (e < E) ? order_key(bias ? l[e] + bias[e] : l[e]) : 0u;
    }
    int sel_e = 0;
    for (int j = 0; j < k; ++j) {
        uint32_t m;
        const int e = warp_select<PER>(key, lane, m);
        if (lane == j) sel_e = e;
    }
    const float sc = (lane < k) ? 1.f / (1.f + expf(-l[sel_e])) : 0.f;
    float sum = 0.f;
    for (int j = 0; j < k; ++j) sum = sum + __shfl_sync(0xffffffffu, sc, j);
    if (lane < k) {
        topk_idx[(size_t)warp * k + lane] = sel_e;
        topk_s[(size_t)warp * k + lane] = sc;
        topk_w[(size_t)warp * k + lane] = sc / sum;
    }
}

// Loss-free bias controller (Table 29): one thread per expert; the total is the sum of the counts.
__global__ void bias_update_kernel(const int32_t *__restrict__ counts, float *__restrict__ bias, int E, int mode, float gamma,
                                   float cap_hi, float cap_lo) {
    __shared__ float s_tot[32];
    float part = 0.f;
    for (int e = threadIdx.x; e < E; e += blockDim.x) part += (float)counts[e];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) part += __shfl_xor_sync(0xffffffffu, part, off);
    if (threadIdx.x % 32 == 0) s_tot[threadIdx.x / 32] = part;
    __syncthreads();
    float total = 0.f;
    for (int w = 0; w < (int)blockDim.x / 32; ++w) total += s_tot[w];
    const float tau = 1.f / (float)E;
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        const float load = total > 0.f ? (float)counts[e] / total : 0.f;
        const float err = tau - load;
        float delta = gamma * (err > 0.f ? 1.f : (err < 0.f ? -1.f : 0.f));
        if (mode == 1) {
            const float lo = cap_lo > 0.f ? cap_lo : tau * tau / cap_hi;
            if (load > cap_hi) { const float z = (load - cap_hi) / tau; delta = -gamma * (1.f + z * z); }
            else if (load < lo) { const float z = (lo - load) / tau; delta = gamma * (1.f + z * z); }
        }
        bias[e] += delta;
    }
}

// Picks the tile: the large one (96 x 96) unless it cannot fill the SMs (few tokens or few experts).
static void launch_logits(const bf16 *X, const float *W_r, const float *bias, float *logits, int T, int d, int E, int num_sms,
                          cudaStream_t s) {
    const long big = (long)((T + 95) / 96) * ((E + 95) / 96);
    if (big >= 2L * num_sms) {
        route_logits_kernel<12, 6><<<dim3((T + 95) / 96, (E + 95) / 96), 128, 0, s>>>(X, W_r, bias, logits, T, d, E);
    } else {
        route_logits_kernel<4, 4><<<dim3((T + 31) / 32, (E + 63) / 64), 128, 0, s>>>(X, W_r, bias, logits, T, d, E);
    }
}

tqp_status launch_route_sigmoid(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *select_bias, int32_t *topk_idx,
                                float *topk_w, float *topk_s, float *logits, cudaStream_t s) {
    const int d = c->desc.d, E = c->desc.E, k = c->desc.k;
    launch_logits(X, W_r, nullptr, logits, T, d, E, c->num_sms, s);
    TQP_LAUNCH_OK(c);
#define TQP_TOPK(P) route_topk_sigmoid_kernel<P><<<(T + 3) / 4, 128, 0, s>>>(logits, select_bias, topk_idx, topk_w, topk_s, T, E, k)
    if (E <= 64) TQP_TOPK(2); else if (E <= 128) TQP_TOPK(4); else if (E <= 256) TQP_TOPK(8); else if (E <= 512) TQP_TOPK(16); else TQP_TOPK(32);
#undef TQP_TOPK
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

tqp_status launch_bias_update(tqp_ctx *c, const int32_t *counts, float *bias, int mode, float gamma, float cap_hi, float cap_lo,
                              cudaStream_t s) {
    bias_update_kernel<<<1, 256, 0, s>>>(counts, bias, c->desc.E, mode, gamma, cap_hi, cap_lo);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

tqp_status launch_route(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *bias, int32_t *topk_idx,
                        float *topk_w, float *logits, cudaStream_t s) {
    const int d = c->desc.d, E = c->desc.E, k = c->desc.k;
    launch_logits(X, W_r, bias, logits, T, d, E, c->num_sms, s);
    TQP_LAUNCH_OK(c);
#define TQP_TOPK(P) route_topk_kernel<P><<<(T + 3) / 4, 128, 0, s>>>(logits, topk_idx, topk_w, T, E, k)
    if (E <= 64) TQP_TOPK(2); else if (E <= 128) TQP_TOPK(4); else if (E <= 256) TQP_TOPK(8); else if (E <= 512) TQP_TOPK(16); else TQP_TOPK(32);
#undef TQP_TOPK
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
