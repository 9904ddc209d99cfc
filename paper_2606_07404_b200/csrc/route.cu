// Router: fp32 logits in the canonical order (R1) + warp-level top-k + softmax over the selected.
// PAPER.md L224 (routing logits + per-expert bias), L239 (top-k over real experts); BASELINE.json configs[0]
// (softmax over the selected logits, ties -> lower expert id).
#include "common.cuh"
#include "tc_ptx.cuh"

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
                                                              int T, int d, int E, const int *__restrict__ gate) {
    if (gate && *gate == 0) return;   // fallback launch behind the screened router: runs only if its self-check tripped
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
                                                         float *__restrict__ topk_w, int T, int E, int k,
                                                         const int *__restrict__ gate) {
    if (gate && *gate == 0) return;
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
                                                                 float *__restrict__ topk_s, int T, int E, int k, const int *__restrict__ gate) {
    if (gate && *gate == 0) return;
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
                          cudaStream_t s, const int *gate = nullptr) {
    const long big = (long)((T + 95) / 96) * ((E + 95) / 96);
    if (big >= 2L * num_sms) {
        route_logits_kernel<12, 6><<<dim3((T + 95) / 96, (E + 95) / 96), 128, 0, s>>>(X, W_r, bias, logits, T, d, E, gate);
    } else {
        route_logits_kernel<4, 4><<<dim3((T + 31) / 32, (E + 63) / 64), 128, 0, s>>>(X, W_r, bias, logits, T, d, E, gate);
    }
}

tqp_status launch_route_sigmoid(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *select_bias, int32_t *topk_idx,
                                float *topk_w, float *topk_s, float *logits, cudaStream_t s, const int *gate) {
    const int d = c->desc.d, E = c->desc.E, k = c->desc.k;
    launch_logits(X, W_r, nullptr, logits, T, d, E, c->num_sms, s, gate);
    TQP_LAUNCH_OK(c);
#define TQP_TOPK(P) route_topk_sigmoid_kernel<P><<<(T + 3) / 4, 128, 0, s>>>(logits, select_bias, topk_idx, topk_w, topk_s, T, E, k, gate)
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
                        float *topk_w, float *logits, cudaStream_t s, const int *gate) {
    const int d = c->desc.d, E = c->desc.E, k = c->desc.k;
    launch_logits(X, W_r, bias, logits, T, d, E, c->num_sms, s, gate);
    TQP_LAUNCH_OK(c);
#define TQP_TOPK(P) route_topk_kernel<P><<<(T + 3) / 4, 128, 0, s>>>(logits, topk_idx, topk_w, T, E, k, gate)
    if (E <= 64) TQP_TOPK(2); else if (E <= 128) TQP_TOPK(4); else if (E <= 256) TQP_TOPK(8); else if (E <= 512) TQP_TOPK(16); else TQP_TOPK(32);
#undef TQP_TOPK
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// =========================================================================================================
// Screened router: the same topk_idx / topk_w as launch_route, bit for bit, at a fraction of the fp32 work.
//
// R1 fixes the value of a logit as one sequential fmaf chain, which the tensor cores cannot reproduce.  But only the k
// selected logits of a token (and the order among them) ever leave the router, so the dense product need not be exact:
//   1. a[t][e] ~ logit[t][e] on the tensor cores (tcgen05, bf16 x (hi + lo) split of W_r, fp32 accumulation), with a bound
//      |a - logit| <= delta_t  (below);
//   2. tau = the k-th largest a[t][.]; at least k experts have logit >= tau - delta_t, so an expert with
//      a < tau - 2 delta_t has logit < tau - delta_t and cannot be among the k largest (strictly: no tie either);
//   3. the remaining candidates (k plus a few) get the canonical chain; top-k, tie-break and softmax run on those exact
//      values with the code of route_topk_kernel.
// delta_t = cK |x_t| max_e |w_e|  (+ 2^-22 max_e |a + bias| when a bias is added), cK = (d 2^-21 + 2^-16) * 1.01:
//   * chain against the real sum: <= d 2^-24 S, S = sum_i |x_i w_i| <= |x_t| |w_e| (Cauchy-Schwarz);
//   * W_r = hi + lo + rest, |rest| <= 2^-16 |w|: the products x hi, x lo are exact in fp32, the dropped part is <= 2^-16 S;
//   * tensor-core accumulation of the 2d exact products: a truncating fp32 adder loses <= 2^-23 of a partial sum per
//     addend, <= 2d 2^-23 S in all; the bound used is twice that, d 2^-21 S (the adder tree inside one MMA is not documented).
// Self-check: every candidate has both values, and |a - logit| <= delta_t / 2 is asserted for each (120 k samples per call
// at cfg 2, typical ratio 1e-3).  A violation, or a token with more than RS_CMAX candidates (e.g. an all-zero row: every
// expert ties), raises a device flag, and the dense exact kernels, launched behind the screen with that flag as their gate,
// recompute the call.  Either way the caller sees the canonical result.
// =========================================================================================================
constexpr int RS_BM = 128, RS_BN = 256, RS_BK = 64, RS_STAGES = 4;
constexpr int RS_A_BYTES = RS_BM * RS_BK * 2, RS_B_BYTES = RS_BN * RS_BK * 2, RS_STAGE_BYTES = RS_A_BYTES + RS_B_BYTES;
constexpr int RS_TC_SMEM = RS_STAGES * RS_STAGE_BYTES + 1024 + 256;
constexpr int RS_CMAX = 64;   // candidates per token held by the screen (two per lane)
constexpr int RS_ROWS = 24, RS_KC = 64, RS_LD = RS_KC + 4;   // candidate rows per chain batch, columns per chunk, floats per tile row
constexpr int RS_WARP_SMEM = 2 * RS_ROWS * RS_LD * 4 + 2 * RS_KC * 2 + 2 * RS_CMAX * 4;   // + RS_CMAX * 4 in the sigmoid variant   // per warp of route_screen_kernel

// W_r [d][E] fp32 -> WrT [E][d] fp32 (rows of the candidate chains) and WrHL [E][2d] bf16 (hi | lo, K-major MMA operand)
__global__ void __launch_bounds__(256) route_prep_kernel(const float *__restrict__ W_r, float *__restrict__ WrT, bf16 *__restrict__ WrHL,
                                                         int *__restrict__ flag, int d, int E) {
    __shared__ float tile[32][33];
    const int i0 = blockIdx.x * 32, e0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int i = i0 + r, e = e0 + threadIdx.x;
        tile[r][threadIdx.x] = (i < d && e < E) ? W_r[(size_t)i * E + e] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int e = e0 + r, i = i0 + threadIdx.x;
        if (e < E && i < d) {
            const float w = tile[threadIdx.x][r];
            const bf16 hi = __float2bfloat16_rn(w);
            const bf16 lo = __float2bfloat16_rn(w - __bfloat162float(hi));   // the difference is exact in fp32
            WrT[(size_t)e * d + i] = w;
            WrHL[(size_t)e * 2 * d + i] = hi;
            WrHL[(size_t)e * 2 * d + d + i] = lo;
        }
    }
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0 && threadIdx.y == 0) *flag = 0;
}

// wn[e] >= |w_e|_2 (one warp per expert; fixed summation order)
__global__ void __launch_bounds__(128) route_wnorm_kernel(const float *__restrict__ WrT, float *__restrict__ wn, int d, int E) {
    const int e = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (e >= E) return;
    float ss = 0.f;
    for (int i = lane; i < d; i += 32) { const float w = WrT[(size_t)e * d + i]; ss = fmaf(w, w, ss); }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, off);
    if (lane == 0) wn[e] = sqrtf(ss) * 1.001f;
}

// a[t][e] = sum_i x[t][i] (hi[e][i] + lo[e][i]): one CTA per 128 tokens x 256 experts, K' = 2d in 64-wide stages (the X tile
// is fetched once for the hi half and once for the lo half of K').  warp 0 TMA, warp 1 MMA issue, warps 2-5 epilogue.
__global__ void __launch_bounds__(192) route_tc_logits_kernel(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapW,
                                                              float *__restrict__ A, int T, int d, int E) {
    using namespace ptx;
    extern __shared__ uint8_t rs_smem[];
    const uint32_t base = (smem_u32(rs_smem) + 1023u) & ~1023u;
    const uint32_t bars = base + RS_STAGES * RS_STAGE_BYTES;
    const uint32_t full0 = bars, empty0 = bars + 8 * RS_STAGES, acc_full = bars + 16 * RS_STAGES, slot = acc_full + 8;
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int t0 = blockIdx.x * RS_BM, e0 = blockIdx.y * RS_BN;
    const int n_mma = min(RS_BN, (E - e0 + 15) & ~15);
    const int nkb = 2 * d / RS_BK;
    if (threadIdx.x == 0) {
        for (int s = 0; s < RS_STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        mbar_init(acc_full, 1);
        mbar_init_fence();
    }
    if (warp == 1) tmem_alloc<1>(slot, RS_BN);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t d_tmem = lds32(slot);

    if (warp == 0) {
        if (elect_one()) {
            Pipe p;
            for (int kb = 0; kb < nkb; ++kb) {
                mbar_wait(empty0 + 8 * p.s, p.ph ^ 1);
                const uint32_t a_s = base + p.s * RS_STAGE_BYTES, b_s = a_s + RS_A_BYTES;
                mbar_expect_tx(full0 + 8 * p.s, RS_STAGE_BYTES);
                int kx = kb * RS_BK;
                if (kx >= d) kx -= d;
                tma_load_2d(a_s, &mapX, kx, t0, full0 + 8 * p.s);
                tma_load_2d(b_s, &mapW, kb * RS_BK, e0, full0 + 8 * p.s);
                p.next(RS_STAGES);
            }
        }
    } else if (warp == 1) {
        if (elect_one()) {
            const uint32_t idesc = make_idesc(RS_BM, n_mma, 0);
            const uint32_t hi_k = desc_hi(1024), lo_k = desc_lo_const(16);   // K-major SW128: SBO = 8 rows x 128 B
            Pipe p;
            for (int kb = 0; kb < nkb; ++kb) {
                mbar_wait(full0 + 8 * p.s, p.ph);
                tc_fence_after();
                const uint32_t a16 = (base + p.s * RS_STAGE_BYTES) >> 4, b16 = a16 + (RS_A_BYTES >> 4);
#pragma unroll
                for (int kk = 0; kk < RS_BK / 16; ++kk)
                    umma_bf16<1>(d_tmem, desc_from(hi_k, lo_k, a16 + kk * 2), desc_from(hi_k, lo_k, b16 + kk * 2), idesc, (kb | kk) != 0);
                umma_commit(empty0 + 8 * p.s);
                p.next(RS_STAGES);
            }
            umma_commit(acc_full);
        }
    } else {
        mbar_wait(acc_full, 0);
        tc_fence_after();
        const int q = warp % 4;                      // the TMEM lane quarter this warp may read
        const int t = t0 + q * 32 + lane;
        float *row = A + (size_t)t * E + e0;
        const bool vec = (E % 4) == 0;
        for (int c0 = 0; c0 < n_mma; c0 += 16) {
            uint32_t v[16];
            tmem_ld16(d_tmem + ((uint32_t)(q * 32) << 16) + c0, v);
            tmem_ld_wait();
            if (t < T) {
                if (vec && e0 + c0 + 16 <= E) {
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        *reinterpret_cast<uint4 *>(row + c0 + 4 * j) = make_uint4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
                } else {
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (e0 + c0 + j < E) row[c0 + j] = __uint_as_float(v[j]);
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<1>(d_tmem, RS_BN);
}

// One warp per token: candidates from the approximate logits, canonical chains for them, exact top-k + softmax.
// SIG: the paper-faithful variant (route_topk_sigmoid_kernel): selection by logit + bias, gate = sigmoid of the UNBIASED logit
// normalised over the selected set, topk_s = the sigmoid values.
template <int PER, bool SIG>
__global__ void __launch_bounds__(128) route_screen_kernel(const float *__restrict__ A, const bf16 *__restrict__ X, const float *__restrict__ WrT,
                                                           const float *__restrict__ wn, const float *__restrict__ bias,
                                                           int32_t *__restrict__ topk_idx, float *__restrict__ topk_w, float *__restrict__ topk_s,
                                                           int *__restrict__ flag, int T, int d, int E, int k, float cK, float chk) {
    extern __shared__ __align__(16) uint8_t rs_sm[];
    const int wib = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int t = blockIdx.x * 4 + wib;
    if (t >= T) return;   // warp-uniform; nothing below synchronises the block
    uint8_t *wsm = rs_sm + (size_t)wib * (RS_WARP_SMEM + (SIG ? RS_CMAX * 4 : 0));
    const uint32_t tile_s = ptx::smem_u32(wsm);                       // [2][RS_ROWS][RS_LD] fp32 (rows padded by 16 bytes: conflict-free)
    const uint32_t xb_s = tile_s + 2 * RS_ROWS * RS_LD * 4;          // [2][RS_KC] bf16: the token's chunk as it comes from X
    int *cl_e = reinterpret_cast<int *>(wsm + 2 * RS_ROWS * RS_LD * 4 + 2 * RS_KC * 2);
    float *cl_v = reinterpret_cast<float *>(cl_e + RS_CMAX);         // approximate value, replaced by the exact one
    float *cl_u = cl_v + RS_CMAX;                                    // SIG: the exact logit without the bias

    // |x_t|^2
    float ss = 0.f;
    {
        const uint4 *xr = reinterpret_cast<const uint4 *>(X + (size_t)t * d);
        for (int c = lane; c < d / 8; c += 32) {
            const uint4 u = xr[c];
            const float2 f0 = bf16x2_to_float2(u.x), f1 = bf16x2_to_float2(u.y), f2 = bf16x2_to_float2(u.z), f3 = bf16x2_to_float2(u.w);
            ss = fmaf(f0.x, f0.x, ss); ss = fmaf(f0.y, f0.y, ss); ss = fmaf(f1.x, f1.x, ss); ss = fmaf(f1.y, f1.y, ss);
            ss = fmaf(f2.x, f2.x, ss); ss = fmaf(f2.y, f2.y, ss); ss = fmaf(f3.x, f3.x, ss); ss = fmaf(f3.y, f3.y, ss);
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, off);
    }
    // approximate logits (+ bias), their keys, the largest magnitude and the largest expert norm
    float v[PER];
    uint32_t key[PER];
    float vmax = 0.f, wmax = 0.f;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        const int e = q * 32 + lane;
        if (e < E) {
            float a = A[(size_t)t * E + e];
            if (bias) a = a + bias[e];
            v[q] = a;
            key[q] = order_key(a);
            vmax = fmaxf(vmax, fabsf(a));
            wmax = fmaxf(wmax, wn[e]);
        } else {
            v[q] = 0.f;
            key[q] = 0u;
        }
    }
    vmax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(vmax)));   // non-negative floats order like their bits
    wmax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(wmax)));
    // tau = k-th largest approximate value
    float tau;
    {
        uint32_t k2[PER];
#pragma unroll
        for (int q = 0; q < PER; ++q) k2[q] = key[q];
        uint32_t m = 0;
        for (int j = 0; j < k; ++j) warp_select<PER>(k2, lane, m);
        tau = key_value(m);
    }
    const float delta = cK * (sqrtf(ss) * 1.001f) * wmax + (bias ? 2.4e-7f * vmax : 0.f);
    const float thr = tau - 2.f * delta - 1e-6f * fabsf(tau);
    // candidate list
    int count = 0;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        const bool c = key[q] != 0u && v[q] >= thr;
        const uint32_t mask = __ballot_sync(0xffffffffu, c);
        if (c) {
            const int pos = count + __popc(mask & ((1u << lane) - 1u));
            if (pos < RS_CMAX) { cl_e[pos] = q * 32 + lane; cl_v[pos] = v[q]; }
        }
        count += __popc(mask);
    }
    bool bad = count > RS_CMAX || count < k;   // count < k: NaN / Inf logits, the dense kernels define what happens then
    if (count > RS_CMAX) count = RS_CMAX;
    __syncwarp();
    // canonical chains (R1): acc = fmaf(x_i, W_r[i][e], acc), i ascending, then + bias.  Lane = candidate; the
    // candidates' rows of W_r^T come in 64-column chunks, two rows per warp-wide cp.async (a half-warp covers 256 contiguous
    // bytes; a lane streaming its own row with 16-byte loads costs one L1 tag cycle per lane and load: 376 us at cfg 2),
    // double-buffered in shared memory; the token's bf16 chunk rides along and is widened in the lane (a shift / a mask).
    constexpr int LPR = RS_KC / 4, RPI = 32 / LPR;   // lanes per row chunk (16 bytes each), rows per warp-wide cp.async
    const int sub = lane / LPR, q = lane % LPR;
    for (int b = 0; b < count; b += RS_ROWS) {
        const int nb = min(RS_ROWS, count - b);
        // row RPI r + sub: its chunk column in W_r^T (advanced by two chunks per trip) and its place in buffer 0
        const float *gp[RS_ROWS / RPI];
        bool on[RS_ROWS / RPI];
#pragma unroll
        for (int r = 0; r < RS_ROWS / RPI; ++r) {
            const int row = RPI * r + sub;
            on[r] = RPI * r < nb;   // warp-uniform: past nb the last group fetches the last candidate's row again
            gp[r] = WrT + (size_t)(on[r] ? cl_e[b + min(row, nb - 1)] : 0) * d + q * 4;
        }
        const uint32_t dst0 = tile_s + (uint32_t)(sub * RS_LD * 4 + q * 16);
        const bf16 *xp = X + (size_t)t * d + lane * 8;
        const uint32_t rowa = tile_s + (uint32_t)(lane * RS_LD * 4);
        float acc = 0.f;
#define RS_ISSUE(BUF, OFF)                                                                                                         \
    do {                                                                                                                           \
        _Pragma("unroll") for (int r = 0; r < RS_ROWS / RPI; ++r) if (on[r])                                                       \
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst0 + (uint32_t)(((BUF) * RS_ROWS + RPI * r) * RS_LD * 4)), \
                         "l"(gp[r] + (OFF)) : "memory");                                                                           \
        if (lane < RS_KC / 8)                                                                                                      \
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(xb_s + (BUF) * RS_KC * 2 + lane * 16), "l"(xp + (OFF)) : "memory"); \
        asm volatile("cp.async.commit_group;" ::: "memory");                                                                       \
    } while (0)
#define RS_CHUNK(BUF)                                                                                                              \
    do {                                                                                                                           \
        __syncwarp();                                                                                                              \
        if (lane < nb) {                                                                                                           \
            _Pragma("unroll") for (int j = 0; j < RS_KC / 8; ++j) {   /* 8 bf16 of x (widened in the lane: a shift / a mask) x 8 of the row */ \
                const uint4 xu = ptx::lds128(xb_s + (uint32_t)((BUF) * RS_KC * 2 + j * 16));                                       \
                const uint4 w0 = ptx::lds128(rowa + (uint32_t)((BUF) * RS_ROWS * RS_LD * 4 + j * 32));                              \
                const uint4 w1 = ptx::lds128(rowa + (uint32_t)((BUF) * RS_ROWS * RS_LD * 4 + j * 32 + 16));                         \
                acc = fmaf(__uint_as_float(xu.x << 16), __uint_as_float(w0.x), acc);                                               \
                acc = fmaf(__uint_as_float(xu.x & 0xffff0000u), __uint_as_float(w0.y), acc);                                       \
                acc = fmaf(__uint_as_float(xu.y << 16), __uint_as_float(w0.z), acc);                                               \
                acc = fmaf(__uint_as_float(xu.y & 0xffff0000u), __uint_as_float(w0.w), acc);                                       \
                acc = fmaf(__uint_as_float(xu.z << 16), __uint_as_float(w1.x), acc);                                               \
                acc = fmaf(__uint_as_float(xu.z & 0xffff0000u), __uint_as_float(w1.y), acc);                                       \
                acc = fmaf(__uint_as_float(xu.w << 16), __uint_as_float(w1.z), acc);                                               \
                acc = fmaf(__uint_as_float(xu.w & 0xffff0000u), __uint_as_float(w1.w), acc);                                       \
            }                                                                                                                      \
        }                                                                                                                          \
        __syncwarp();                                                                                                              \
    } while (0)
        // two chunks per trip (d % 128 == 0), so that the buffer index is a compile-time constant
        RS_ISSUE(0, 0);
        for (int i0 = 0; i0 < d; i0 += 2 * RS_KC) {
            RS_ISSUE(1, RS_KC);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            RS_CHUNK(0);
#pragma unroll
            for (int r = 0; r < RS_ROWS / 2; ++r) gp[r] += 2 * RS_KC;
            xp += 2 * RS_KC;
            if (i0 + 2 * RS_KC < d) {
                RS_ISSUE(0, 0);
                asm volatile("cp.async.wait_group 1;" ::: "memory");
            } else {
                asm volatile("cp.async.wait_group 0;" ::: "memory");
            }
            RS_CHUNK(1);
        }
#undef RS_ISSUE
#undef RS_CHUNK
        if (lane < nb) {
            const int e = cl_e[b + lane];
            if (SIG) cl_u[b + lane] = acc;
            if (bias) acc = acc + bias[e];
            if (!(fabsf(acc - cl_v[b + lane]) <= chk * delta)) bad = true;   // cl_v held the approximate value until here
            cl_v[b + lane] = acc;
        }
    }
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicExch(flag, 1);
    __syncwarp();
    // exact top-k among the candidates under (-logit, id)
    uint32_t ck[2];
    int ce[2];
#pragma unroll
    for (int s2 = 0; s2 < 2; ++s2) {
        const int idx = s2 * 32 + lane;
        ck[s2] = idx < count ? order_key(cl_v[idx]) : 0u;
        ce[s2] = idx < count ? cl_e[idx] : 0x7fffffff;
    }
    float sel_l = 0.f;
    int sel_e = 0;
    for (int j = 0; j < k; ++j) {
        const uint32_t m = __reduce_max_sync(0xffffffffu, max(ck[0], ck[1]));
        int cand = 0x7fffffff;
        if (ck[1] == m) cand = ce[1];
        if (ck[0] == m) cand = min(cand, ce[0]);
        const int e = __reduce_min_sync(0xffffffffu, cand);   // ties -> lower expert id
        float u = 0.f;   // SIG: the winner's unbiased logit, from the lane that holds it
        if (SIG) {
            const float mine = ce[0] == e ? cl_u[lane] : ce[1] == e ? cl_u[32 + lane] : 0.f;
            const uint32_t own = __ballot_sync(0xffffffffu, ce[0] == e || ce[1] == e);
            u = __shfl_sync(0xffffffffu, mine, __ffs(own) - 1);
        }
        if (ce[0] == e) ck[0] = 0u;
        if (ce[1] == e) ck[1] = 0u;
        if (lane == j) { sel_l = SIG ? u : key_value(m); sel_e = e; }
    }
    if (SIG) {
        const float sc = (lane < k) ? 1.f / (1.f + expf(-sel_l)) : 0.f;
        float ssum = 0.f;
        for (int j = 0; j < k; ++j) ssum = ssum + __shfl_sync(0xffffffffu, sc, j);
        if (lane < k) {
            topk_idx[(size_t)t * k + lane] = sel_e;
            topk_s[(size_t)t * k + lane] = sc;
            topk_w[(size_t)t * k + lane] = sc / ssum;
        }
        return;
    }
    const float m0 = __shfl_sync(0xffffffffu, sel_l, 0);
    const float ex = (lane < k) ? expf(sel_l - m0) : 0.f;
    float sum = 0.f;
    for (int j = 0; j < k; ++j) sum = sum + __shfl_sync(0xffffffffu, ex, j);
    if (lane < k) {
        topk_idx[(size_t)t * k + lane] = sel_e;
        topk_w[(size_t)t * k + lane] = ex / sum;
    }
}

// forced: wherever the kernels can run.  Otherwise also where it pays: the dense chain costs T E d FMAs at ~ 22 T/s, the
// screen ~ 50 us of fixed work plus 4 d bytes of L2 traffic for each of a token's k + (a few) candidate rows at ~ 7 TB/s
// (measured: cfg 1 57 us dense / 106 us screened, cfg 2 432 / 244 us).
bool route_screen_applicable(const tqp_ctx *c, int T, bool forced) {
    const tqp_layer_desc &D = c->desc;
    if (!(D.d % 128 == 0 && D.E <= 1024 && D.k <= 32 && D.k <= D.E)) return false;
    if (forced) return true;
    return D.E > 6 * (D.k + 4) && (double)T * D.E * D.d >= 3.0e9;
}

tqp_status launch_route_screened(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *bias, int32_t *topk_idx,
                                 float *topk_w, float *topk_s, const CUtensorMap *mapX, const CUtensorMap *mapW, cudaStream_t s) {
    const bool sig = topk_s != nullptr;
    const int d = c->desc.d, E = c->desc.E, k = c->desc.k;
    float *WrT = c->p<float>(c->ws.WrT), *wn = c->p<float>(c->ws.wnorm), *A = c->p<float>(c->ws.logits);
    bf16 *WrHL = c->p<bf16>(c->ws.WrHL);
    int *flag = c->p<int>(c->ws.rflag);
    route_prep_kernel<<<dim3((d + 31) / 32, (E + 31) / 32), dim3(32, 8), 0, s>>>(W_r, WrT, WrHL, flag, d, E);
    TQP_LAUNCH_OK(c);
    route_wnorm_kernel<<<(E + 3) / 4, 128, 0, s>>>(WrT, wn, d, E);
    TQP_LAUNCH_OK(c);
    if (tqp_status st = ensure_dyn_smem(c, reinterpret_cast<const void *>(&route_tc_logits_kernel), RS_TC_SMEM)) return st;
    route_tc_logits_kernel<<<dim3((T + RS_BM - 1) / RS_BM, (E + RS_BN - 1) / RS_BN), 192, RS_TC_SMEM, s>>>(*mapX, *mapW, A, T, d, E);
    TQP_LAUNCH_OK(c);
    const float cK = ((float)d * 4.76837158e-7f + 1.52587891e-5f) * 1.01f;   // d 2^-21 + 2^-16
    const float chk = c->route_impl == 3 ? -1.f : 0.5f;
    const int smem = 4 * (RS_WARP_SMEM + (sig ? RS_CMAX * 4 : 0));
#define TQP_SCREEN(P)                                                                                                     \
    do {                                                                                                                  \
        if (sig) {                                                                                                        \
            if (tqp_status st = ensure_dyn_smem(c, reinterpret_cast<const void *>(&route_screen_kernel<P, true>), smem)) return st; \
            route_screen_kernel<P, true><<<(T + 3) / 4, 128, smem, s>>>(A, X, WrT, wn, bias, topk_idx, topk_w, topk_s, flag, T, d, E, k, cK, chk); \
        } else {                                                                                                          \
            if (tqp_status st = ensure_dyn_smem(c, reinterpret_cast<const void *>(&route_screen_kernel<P, false>), smem)) return st; \
            route_screen_kernel<P, false><<<(T + 3) / 4, 128, smem, s>>>(A, X, WrT, wn, bias, topk_idx, topk_w, nullptr, flag, T, d, E, k, cK, chk); \
        }                                                                                                                 \
    } while (0)
    if (E <= 64) TQP_SCREEN(2); else if (E <= 128) TQP_SCREEN(4); else if (E <= 256) TQP_SCREEN(8); else if (E <= 512) TQP_SCREEN(16); else TQP_SCREEN(32);
#undef TQP_SCREEN
    TQP_LAUNCH_OK(c);
    // the dense exact kernels behind the flag: two empty launches unless the self-check tripped
    if (sig) return launch_route_sigmoid(c, T, X, W_r, bias, topk_idx, topk_w, topk_s, A, s, flag);
    return launch_route(c, T, X, W_r, bias, topk_idx, topk_w, A, s, flag);
}

}  // namespace tqp
