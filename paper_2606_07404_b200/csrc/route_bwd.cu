// Router backward with the selection held constant (the router is trained):
//   dl_j = w_j (dw_j - sum_i w_i dw_i);  dX[t] += sum_j dl_j W_r[:,e_j];  dW_r[:,e] = sum_{rows of e} X[t] dl.
// dW_r is reduced per expert over the rows of the dispatch permutation in ascending order (deterministic).
#include "common.cuh"

namespace tqp {

// sc == nullptr: softmax over the selected logits.  sc != nullptr: normalised sigmoid scores (tqp_route_sigmoid):
// dl_j = (dw_j - sum_i w_i dw_i) w_j (1 - s_j).
__global__ void route_dl_kernel(const float *__restrict__ w, const float *__restrict__ dw, const float *__restrict__ sc,
                                float *__restrict__ dl, int T, int k) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    float dotp = 0.f;
    for (int j = 0; j < k; ++j) dotp = fmaf(w[(size_t)t * k + j], dw[(size_t)t * k + j], dotp);
    for (int j = 0; j < k; ++j) {
        float g = w[(size_t)t * k + j] * (dw[(size_t)t * k + j] - dotp);
        if (sc) g *= 1.f - sc[(size_t)t * k + j];
        dl[(size_t)t * k + j] = g;
    }
}

__global__ void transpose_wr_kernel(const float *__restrict__ W_r, float *__restrict__ WrT, int d, int E) {
    __shared__ float tile[32][33];
    int i0 = blockIdx.x * 32, e0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += 8) {
        int i = i0 + r, e = e0 + threadIdx.x;
        tile[r][threadIdx.x] = (i < d && e < E) ? W_r[(size_t)i * E + e] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        int e = e0 + r, i = i0 + threadIdx.x;
        if (e < E && i < d) WrT[(size_t)e * d + i] = tile[threadIdx.x][r];
    }
}

// dX[t][col..col+8) += sum_j dl[t][j] * WrT[e_j][col..]
__global__ void __launch_bounds__(256) route_dx_kernel(const float *__restrict__ WrT, const int32_t *__restrict__ topk_idx,
                                                       const float *__restrict__ dl, bf16 *__restrict__ dX, int T, int d, int k) {
    const int slabs = (d + 255) / 256;
    const int gw = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
    const int t = gw / slabs, slab = gw % slabs;
    if (t >= T) return;
    const int col = slab * 256 + lane * 8;
    if (col >= d) return;
    uint4 cur = *reinterpret_cast<const uint4 *>(dX + (size_t)t * d + col);
    const uint32_t *cp = reinterpret_cast<const uint32_t *>(&cur);
    float acc[8];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        float2 f = bf16x2_to_float2(cp[q]);
        acc[2 * q] = f.x;
        acc[2 * q + 1] = f.y;
    }
    for (int j = 0; j < k; ++j) {
        const int e = topk_idx[(size_t)t * k + j];
        const float g = dl[(size_t)t * k + j];
        const float4 *wr = reinterpret_cast<const float4 *>(WrT + (size_t)e * d + col);
        float4 a = wr[0], b = wr[1];
        acc[0] = fmaf(g, a.x, acc[0]); acc[1] = fmaf(g, a.y, acc[1]); acc[2] = fmaf(g, a.z, acc[2]); acc[3] = fmaf(g, a.w, acc[3]);
        acc[4] = fmaf(g, b.x, acc[4]); acc[5] = fmaf(g, b.y, acc[5]); acc[6] = fmaf(g, b.z, acc[6]); acc[7] = fmaf(g, b.w, acc[7]);
    }
    uint4 o;
    uint32_t *op = reinterpret_cast<uint32_t *>(&o);
#pragma unroll
    for (int q = 0; q < 4; ++q) op[q] = float2_to_bf16x2(acc[2 * q], acc[2 * q + 1]);
    *reinterpret_cast<uint4 *>(dX + (size_t)t * d + col) = o;
}

// dW_r[i][e] = sum_{p in [offsets[e], offsets[e+1])} X[perm[p]/k][i] * dl[perm[p]];  block = (expert, 512 columns):
// 64 threads x 8 columns (16-byte loads of the gathered X rows, which stay L2-resident), row indices and dl staged
// through shared memory 64 rows at a time, rows in ascending p (deterministic), four rows of loads in flight.
constexpr int DWR_COLS = 512, DWR_CHUNK = 64;
__global__ void __launch_bounds__(64) route_dwr_kernel(const bf16 *__restrict__ X, const float *__restrict__ dl,
                                                       const int32_t *__restrict__ offsets, const int32_t *__restrict__ perm,
                                                       float *__restrict__ dW_r, int d, int E, int k) {
    __shared__ int s_tok[DWR_CHUNK];
    __shared__ float s_dl[DWR_CHUNK];
    const int e = blockIdx.x, col = blockIdx.y * DWR_COLS + threadIdx.x * 8;
    const int p0 = offsets[e], p1 = offsets[e + 1];
    const bool ok = col < d;
    float acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.f;
    for (int pc = p0; pc < p1; pc += DWR_CHUNK) {
        const int n = min(DWR_CHUNK, p1 - pc);
        __syncthreads();
        if ((int)threadIdx.x < n) {
            const int a = perm[pc + threadIdx.x];
            s_tok[threadIdx.x] = a / k;
            s_dl[threadIdx.x] = dl[a];
        }
        __syncthreads();
        if (!ok) continue;
        for (int r0 = 0; r0 < n; r0 += 4) {
            uint4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
                v[u] = (r0 + u < n) ? *reinterpret_cast<const uint4 *>(X + (size_t)s_tok[r0 + u] * d + col) : make_uint4(0, 0, 0, 0);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float g = (r0 + u < n) ? s_dl[r0 + u] : 0.f;
                const uint32_t *vp = reinterpret_cast<const uint32_t *>(&v[u]);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    float2 f = bf16x2_to_float2(vp[q]);
                    acc[2 * q] = fmaf(f.x, g, acc[2 * q]);
                    acc[2 * q + 1] = fmaf(f.y, g, acc[2 * q + 1]);
                }
            }
        }
    }
    if (ok) {
#pragma unroll
        for (int q = 0; q < 8; ++q) dW_r[(size_t)(col + q) * E + e] = acc[q];
    }
}

tqp_status launch_route_bwd(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const int32_t *topk_idx,
                            const float *topk_w, const float *topk_s, const float *dtopk_w, const int32_t *offsets,
                            const int32_t *perm, bf16 *dX, float *dW_r, cudaStream_t s) {
    const int d = c->desc.d, E = c->desc.E, k = c->desc.k;
    float *dl = c->p<float>(c->ws.dl), *WrT = c->p<float>(c->ws.WrT);
    route_dl_kernel<<<(T + 127) / 128, 128, 0, s>>>(topk_w, dtopk_w, topk_s, dl, T, k);
    TQP_LAUNCH_OK(c);
    transpose_wr_kernel<<<dim3((d + 31) / 32, (E + 31) / 32), dim3(32, 8), 0, s>>>(W_r, WrT, d, E);
    TQP_LAUNCH_OK(c);
    const int slabs = (d + 255) / 256;
    const size_t warps = (size_t)T * slabs;
    route_dx_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, s>>>(WrT, topk_idx, dl, dX, T, d, k);
    TQP_LAUNCH_OK(c);
    route_dwr_kernel<<<dim3(E, (d + DWR_COLS - 1) / DWR_COLS), 64, 0, s>>>(X, dl, offsets, perm, dW_r, d, E, k);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
