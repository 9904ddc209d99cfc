// HBM-bound row kernels of the path: permuted-row gather, SwiGLU forward/backward, weighted combine and its
// backward, dispatch backward, codebook -> bf16 LUT.  All use 16-byte vector accesses, one warp per row.
// SURVEY.md §8(a) rows a3, a6, a7, a9, a11; PAPER.md L239 (top-k combine), L401 (gate/up/down).
#include "common.cuh"

namespace tqp {

__device__ __forceinline__ uint4 ld_nc(const uint4 *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

// Xp[p] = X[perm[p] / k]
__global__ void __launch_bounds__(256) gather_rows_kernel(const bf16 *__restrict__ X, const int32_t *__restrict__ perm,
                                                          bf16 *__restrict__ Xp, int N, int d, int k) {
    const int row = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (row >= N) return;
    const int t = perm[row] / k;
    const uint4 *src = reinterpret_cast<const uint4 *>(X + (size_t)t * d);
    uint4 *dst = reinterpret_cast<uint4 *>(Xp + (size_t)row * d);
    for (int v = lane; v < d / 8; v += 32) dst[v] = src[v];
}

// H = silu(G) * U.  Two 16-byte vectors per thread (half a grid apart), all four loads issued before the arithmetic.
__device__ __forceinline__ uint4 swiglu_fwd_vec(const uint4 &g, const uint4 &u) {
    uint4 h;
    const uint32_t *gp = reinterpret_cast<const uint32_t *>(&g), *up = reinterpret_cast<const uint32_t *>(&u);
    uint32_t *hp = reinterpret_cast<uint32_t *>(&h);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        float2 gf = bf16x2_to_float2(gp[q]), uf = bf16x2_to_float2(up[q]);
        float h0 = gf.x / (1.f + __expf(-gf.x)) * uf.x;
        float h1 = gf.y / (1.f + __expf(-gf.y)) * uf.y;
        hp[q] = float2_to_bf16x2(h0, h1);
    }
    return h;
}
__global__ void __launch_bounds__(256) swiglu_fwd_kernel(const uint4 *__restrict__ G, const uint4 *__restrict__ U,
                                                         uint4 *__restrict__ H, size_t nvec, size_t half) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x, i2 = i + half;
    if (i >= half) return;
    const bool two = i2 < nvec;
    const uint4 z = make_uint4(0, 0, 0, 0);
    const uint4 g = ld_nc(G + i), u = ld_nc(U + i), g2 = two ? ld_nc(G + i2) : z, u2 = two ? ld_nc(U + i2) : z;
    H[i] = swiglu_fwd_vec(g, u);
    if (two) H[i2] = swiglu_fwd_vec(g2, u2);
}

// sig = sigmoid(G); dU = dH*G*sig; dG = dH*U*sig*(1+G*(1-sig))
__global__ void __launch_bounds__(256) swiglu_bwd_kernel(const uint4 *__restrict__ dH, const uint4 *__restrict__ G,
                                                         const uint4 *__restrict__ U, uint4 *__restrict__ dG,
                                                         uint4 *__restrict__ dU, size_t nvec) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nvec) return;
    uint4 dh = ld_nc(dH + i), g = ld_nc(G + i), u = ld_nc(U + i), og, ou;
    const uint32_t *dp = reinterpret_cast<const uint32_t *>(&dh), *gp = reinterpret_cast<const uint32_t *>(&g),
                   *up = reinterpret_cast<const uint32_t *>(&u);
    uint32_t *ogp = reinterpret_cast<uint32_t *>(&og), *oup = reinterpret_cast<uint32_t *>(&ou);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        float2 df = bf16x2_to_float2(dp[q]), gf = bf16x2_to_float2(gp[q]), uf = bf16x2_to_float2(up[q]);
        float s0 = 1.f / (1.f + __expf(-gf.x)), s1 = 1.f / (1.f + __expf(-gf.y));
        oup[q] = float2_to_bf16x2(df.x * gf.x * s0, df.y * gf.y * s1);
        ogp[q] = float2_to_bf16x2(df.x * uf.x * s0 * (1.f + gf.x * (1.f - s0)), df.y * uf.y * s1 * (1.f + gf.y * (1.f - s1)));
    }
    dG[i] = og;
    dU[i] = ou;
}

// Y[t] = sum_j w[t][j] * Ye[inv_perm[t*k+j]]   (w == nullptr: plain sum -> dispatch backward).
// One warp per (token, 256-column slab): fp32 accumulate, j ascending.
__global__ void __launch_bounds__(256) combine_kernel(const bf16 *__restrict__ Ye, const int32_t *__restrict__ inv_perm,
                                                      const float *__restrict__ w, bf16 *__restrict__ Y, int T, int d, int k) {
    const int slabs = (d + 255) / 256;
    const int gw = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    const int t = gw / slabs, slab = gw % slabs;
    if (t >= T) return;
    const int col = slab * 256 + lane * 8;
    const bool on = col < d;   // d % 256 == 128: the upper half-warp of the last slab only takes part in the shuffles
    float acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.f;
    // lane j holds the j-th source row and weight (k <= 32); the rows are fetched four at a time (independent loads in flight)
    // and accumulated in ascending j
    const int my_p = lane < k ? inv_perm[(size_t)t * k + lane] : 0;
    const float my_w = (w && lane < k) ? w[(size_t)t * k + lane] : 1.f;
    for (int j0 = 0; j0 < k; j0 += 4) {
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int p = __shfl_sync(0xffffffffu, my_p, (j0 + u) & 31);
            v[u] = (on && j0 + u < k) ? ld_nc(reinterpret_cast<const uint4 *>(Ye + (size_t)p * d + col)) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float wj = __shfl_sync(0xffffffffu, my_w, (j0 + u) & 31);
            if (j0 + u >= k) continue;
            const uint32_t *vp = reinterpret_cast<const uint32_t *>(&v[u]);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                float2 f = bf16x2_to_float2(vp[q]);
                acc[2 * q] = fmaf(wj, f.x, acc[2 * q]);
                acc[2 * q + 1] = fmaf(wj, f.y, acc[2 * q + 1]);
            }
        }
    }
    uint4 o;
    uint32_t *op = reinterpret_cast<uint32_t *>(&o);
#pragma unroll
    for (int q = 0; q < 4; ++q) op[q] = float2_to_bf16x2(acc[2 * q], acc[2 * q + 1]);
    if (on) *reinterpret_cast<uint4 *>(Y + (size_t)t * d + col) = o;
}

// dYe[p] = w[a] * dY[t];  dw[a] = <dY[t], Ye[p]>.  One warp per assignment a.
__global__ void __launch_bounds__(256) combine_bwd_kernel(const bf16 *__restrict__ dY, const bf16 *__restrict__ Ye,
                                                          const int32_t *__restrict__ inv_perm, const float *__restrict__ w,
                                                          bf16 *__restrict__ dYe, float *__restrict__ dw, int N, int d, int k) {
    const int a = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (a >= N) return;
    const int t = a / k, p = inv_perm[a];
    const float wa = w[a];
    const uint4 *src = reinterpret_cast<const uint4 *>(dY + (size_t)t * d);
    const uint4 *ye = reinterpret_cast<const uint4 *>(Ye + (size_t)p * d);
    uint4 *dst = reinterpret_cast<uint4 *>(dYe + (size_t)p * d);
    float dot = 0.f;
    for (int v = lane; v < d / 8; v += 32) {
        uint4 x = src[v], o;
        const uint32_t *xp = reinterpret_cast<const uint32_t *>(&x);
        uint32_t *op = reinterpret_cast<uint32_t *>(&o);
        if (dw) {
            uint4 y = ld_nc(ye + v);
            const uint32_t *yp = reinterpret_cast<const uint32_t *>(&y);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                float2 xf = bf16x2_to_float2(xp[q]), yf = bf16x2_to_float2(yp[q]);
                dot = fmaf(xf.x, yf.x, dot);
                dot = fmaf(xf.y, yf.y, dot);
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            float2 xf = bf16x2_to_float2(xp[q]);
            op[q] = float2_to_bf16x2(wa * xf.x, wa * xf.y);
        }
        dst[v] = o;
    }
    if (dw) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
        if (lane == 0) dw[a] = dot;
    }
}

// dw[a] = <dY[t], Ye[inv_perm[a]]> only (the fused combine-backward writes dYe elsewhere).  One warp per assignment.
__global__ void __launch_bounds__(256) combine_dw_kernel(const bf16 *__restrict__ dY, const bf16 *__restrict__ Ye,
                                                         const int32_t *__restrict__ inv_perm, float *__restrict__ dw,
                                                         int N, int d, int k) {
    const int a = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    if (a >= N) return;
    const int t = a / k, p = inv_perm[a];
    const uint4 *src = reinterpret_cast<const uint4 *>(dY + (size_t)t * d);
    const uint4 *ye = reinterpret_cast<const uint4 *>(Ye + (size_t)p * d);
    float dot = 0.f;
    for (int v = lane; v < d / 8; v += 32) {
        uint4 x = src[v], y = ld_nc(ye + v);
        const uint32_t *xp = reinterpret_cast<const uint32_t *>(&x), *yp = reinterpret_cast<const uint32_t *>(&y);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            float2 xf = bf16x2_to_float2(xp[q]), yf = bf16x2_to_float2(yp[q]);
            dot = fmaf(xf.x, yf.x, dot);
            dot = fmaf(xf.y, yf.y, dot);
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
    if (lane == 0) dw[a] = dot;
}

// bf16 lookup table of the codebook (fp16 -> bf16, RNE), [256][8]
__global__ void make_lut_kernel(const __half *__restrict__ cb, bf16 *__restrict__ lut) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < 256 * 8) lut[i] = __float2bfloat16_rn(__half2float(cb[i]));
}

tqp_status launch_gather_rows(tqp_ctx *c, int N, const bf16 *X, const int32_t *perm, bf16 *Xp, cudaStream_t s) {
    gather_rows_kernel<<<(N + 7) / 8, 256, 0, s>>>(X, perm, Xp, N, c->desc.d, c->desc.k);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
tqp_status launch_swiglu_fwd(tqp_ctx *c, int N, const bf16 *G, const bf16 *U, bf16 *H, cudaStream_t s) {
    const size_t nvec = (size_t)N * c->desc.F / 8, half = (nvec + 1) / 2;
    swiglu_fwd_kernel<<<(unsigned)((half + 255) / 256), 256, 0, s>>>((const uint4 *)G, (const uint4 *)U, (uint4 *)H, nvec, half);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
tqp_status launch_swiglu_bwd(tqp_ctx *c, int N, const bf16 *dH, const bf16 *G, const bf16 *U, bf16 *dG, bf16 *dU,
                             cudaStream_t s) {
    size_t nvec = (size_t)N * c->desc.F / 8;
    swiglu_bwd_kernel<<<(unsigned)((nvec + 255) / 256), 256, 0, s>>>((const uint4 *)dH, (const uint4 *)G, (const uint4 *)U,
                                                                      (uint4 *)dG, (uint4 *)dU, nvec);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
tqp_status launch_combine(tqp_ctx *c, int T, const bf16 *Ye, const int32_t *inv_perm, const float *topk_w, bf16 *Y,
                          cudaStream_t s) {
    const int d = c->desc.d, slabs = (d + 255) / 256;
    const size_t warps = (size_t)T * slabs;
    combine_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, s>>>(Ye, inv_perm, topk_w, Y, T, d, c->desc.k);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
tqp_status launch_combine_bwd(tqp_ctx *c, int T, const bf16 *dY, const bf16 *Ye, const int32_t *inv_perm,
                              const float *topk_w, bf16 *dYe, float *dtopk_w, cudaStream_t s) {
    const int N = T * c->desc.k;
    combine_bwd_kernel<<<(N + 7) / 8, 256, 0, s>>>(dY, Ye, inv_perm, topk_w, dYe, dtopk_w, N, c->desc.d, c->desc.k);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
tqp_status launch_combine_dw(tqp_ctx *c, int T, const bf16 *dY, const bf16 *Ye, const int32_t *inv_perm, float *dtopk_w,
                             cudaStream_t s) {
    const int N = T * c->desc.k;
    combine_dw_kernel<<<(N + 7) / 8, 256, 0, s>>>(dY, Ye, inv_perm, dtopk_w, N, c->desc.d, c->desc.k);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
// fp16 scale -> the bf16 pair (s, s) the backward dequant producers multiply with: frozen weights, so done once at bind time
__global__ void scale_pairs_kernel(const __half *__restrict__ scale, uint32_t *__restrict__ out, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const __nv_bfloat162 v = __float2bfloat162_rn(__half2float(scale[i]));
    out[i] = *reinterpret_cast<const uint32_t *>(&v);
}
tqp_status launch_scale_pairs(tqp_ctx *c, const __half *scale, uint32_t *out, size_t n, cudaStream_t s) {
    scale_pairs_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(scale, out, n);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
tqp_status launch_make_lut(tqp_ctx *c, const __half *codebook, bf16 *lut, cudaStream_t s) {
    make_lut_kernel<<<8, 256, 0, s>>>(codebook, lut);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
