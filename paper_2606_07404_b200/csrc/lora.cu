// Adapter side products of the TQP layer (rank-r adapter on each weight pack, only the adapters train).
//   lora_down : P[p][0..r) = s * in[p][:] . W_e          (x.A, h.A_d forward;  dy.B^T backward)   -> [N][64] bf16
//   lora_wgrad: grad[e]    = sum_{p in e} small[p]^T big[p]  (dA = x^T z, dB = (xA)^T dy), fp32, deterministic
// Both are tall-skinny grouped contractions whose cost is reading the [N][K] operand once from HBM; they use
// warp-level bf16 MMA (wmma) with fp32 accumulation, operands staged through shared memory with row masking
// so rows of a neighbouring expert (or beyond N) never enter a sum.
#include <mma.h>

#include "common.cuh"

namespace tqp {
using namespace nvcuda;

constexpr int LD_KC = 128;            // K-chunk staged per iteration in lora_down
constexpr int LD_LDS = LD_KC + 8;     // padded smem row (bf16)

// grid = (max_tiles, kTileRows/64), block = 128 (4 warps, 16 rows each)
template <int R>
__global__ void __launch_bounds__(128) lora_down_kernel(const bf16 *__restrict__ in, int K, const bf16 *__restrict__ W,
                                                        int w_kr, float s, bf16 *__restrict__ out,
                                                        const Tile *__restrict__ tiles, const int32_t *__restrict__ num_tiles) {
    __shared__ __align__(32) bf16 a_s[4][16][LD_LDS];
    __shared__ __align__(32) float o_s[4][16][R + 4];
    if ((int)blockIdx.x >= *num_tiles) return;
    const Tile t = tiles[blockIdx.x];
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int g = blockIdx.y * 4 + warp;
    if (g * 16 >= t.rows) return;
    const int row0 = t.row0 + g * 16, valid = min(16, t.rows - g * 16);
    const bf16 *We = W + (size_t)t.expert * K * R;
    wmma::fragment<wmma::accumulator, 16, 16, 16, float> acc[R / 16];
#pragma unroll
    for (int n = 0; n < R / 16; ++n) wmma::fill_fragment(acc[n], 0.f);

    for (int k0 = 0; k0 < K; k0 += LD_KC) {
        // stage 16 rows x 128 k, zero rows >= valid.  2 rows per instruction (16 lanes x 16 B each).
#pragma unroll
        for (int it = 0; it < 8; ++it) {
            int r = it * 2 + lane / 16, cv = lane % 16;
            uint4 v = make_uint4(0, 0, 0, 0);
            if (r < valid) v = *reinterpret_cast<const uint4 *>(in + (size_t)(row0 + r) * K + k0 + cv * 8);
            *reinterpret_cast<uint4 *>(&a_s[warp][r][cv * 8]) = v;
        }
        __syncwarp();
#pragma unroll
        for (int kk = 0; kk < LD_KC; kk += 16) {
            wmma::fragment<wmma::matrix_a, 16, 16, 16, bf16, wmma::row_major> af;
            wmma::load_matrix_sync(af, &a_s[warp][0][kk], LD_LDS);
#pragma unroll
            for (int n = 0; n < R / 16; ++n) {
                if (w_kr) {   // W_e[K][R]
                    wmma::fragment<wmma::matrix_b, 16, 16, 16, bf16, wmma::row_major> bfm;
                    wmma::load_matrix_sync(bfm, We + (size_t)(k0 + kk) * R + n * 16, R);
                    wmma::mma_sync(acc[n], af, bfm, acc[n]);
                } else {      // W_e[R][K]  (B^T use)
                    wmma::fragment<wmma::matrix_b, 16, 16, 16, bf16, wmma::col_major> bfm;
                    wmma::load_matrix_sync(bfm, We + (size_t)(n * 16) * K + k0 + kk, K);
                    wmma::mma_sync(acc[n], af, bfm, acc[n]);
                }
            }
        }
        __syncwarp();
    }
#pragma unroll
    for (int n = 0; n < R / 16; ++n) wmma::store_matrix_sync(&o_s[warp][0][n * 16], acc[n], R + 4, wmma::mem_row_major);
    __syncwarp();
    for (int v = lane; v < 16 * R; v += 32) {
        int r = v / R, q = v % R;
        if (r < valid) out[(size_t)(row0 + r) * kLoraPad + q] = __float2bfloat16_rn(s * o_s[warp][r][q]);
    }
}

// r = 8 (config 0): plain CUDA-core version, one warp per row.
__global__ void __launch_bounds__(128) lora_down_small_kernel(const bf16 *__restrict__ in, int K, int R, const bf16 *__restrict__ W,
                                                              int w_kr, float s, bf16 *__restrict__ out,
                                                              const Tile *__restrict__ tiles, const int32_t *__restrict__ num_tiles) {
    if ((int)blockIdx.x >= *num_tiles) return;
    const Tile t = tiles[blockIdx.x];
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const bf16 *We = W + (size_t)t.expert * K * R;
    for (int r = blockIdx.y * 4 + warp; r < t.rows; r += gridDim.y * 4) {
        const bf16 *x = in + (size_t)(t.row0 + r) * K;
        for (int q = 0; q < R; ++q) {
            float acc = 0.f;
            for (int kx = lane; kx < K; kx += 32) {
                float wv = __bfloat162float(w_kr ? We[(size_t)kx * R + q] : We[(size_t)q * K + kx]);
                acc = fmaf(__bfloat162float(x[kx]), wv, acc);
            }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
            if (lane == 0) out[(size_t)(t.row0 + r) * kLoraPad + q] = __float2bfloat16_rn(s * acc);
        }
    }
}

tqp_status launch_lora_down(tqp_ctx *c, const bf16 *in, int K, const bf16 *W, int w_kr, float s, bf16 *out, cudaStream_t st) {
    const Tile *tiles = c->p<Tile>(c->ws.tiles);
    const int32_t *nt = c->p<int32_t>(c->ws.num_tiles);
    dim3 grid(c->max_tiles, kTileRows / 64);
    const int r = c->desc.r;
    if (r == 16) lora_down_kernel<16><<<grid, 128, 0, st>>>(in, K, W, w_kr, s, out, tiles, nt);
    else if (r == 32) lora_down_kernel<32><<<grid, 128, 0, st>>>(in, K, W, w_kr, s, out, tiles, nt);
    else lora_down_small_kernel<<<grid, 128, 0, st>>>(in, K, r, W, w_kr, s, out, tiles, nt);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// ---- weight gradients -----------------------------------------------------------------------------------------
constexpr int WG_P = 32;   // rows per iteration
constexpr int WG_A = 64;   // columns of `big` per block

// grid = (E, width/64), block = 128.  acc tile per warp: [R x 16 a-columns].
template <int R>
__global__ void __launch_bounds__(128) lora_wgrad_kernel(const bf16 *__restrict__ big, int width, const bf16 *__restrict__ small_,
                                                         const int32_t *__restrict__ offsets, int out_ar, float *__restrict__ grad) {
    __shared__ __align__(32) bf16 big_s[WG_P][WG_A + 8];
    __shared__ __align__(32) bf16 sm_s[WG_P][R + 8];
    const int e = blockIdx.x, a0 = blockIdx.y * WG_A;
    const int warp = threadIdx.x / 32, tid = threadIdx.x;
    const int p0 = offsets[e], p1 = offsets[e + 1];
    wmma::fragment<wmma::accumulator, 16, 16, 16, float> acc[R / 16];
#pragma unroll
    for (int n = 0; n < R / 16; ++n) wmma::fill_fragment(acc[n], 0.f);
    for (int p = p0; p < p1; p += WG_P) {
        // big tile: 32 rows x 64 cols = 256 uint4, 2 per thread
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            int v = tid + it * 128, r = v / 8, cv = v % 8;
            uint4 x = make_uint4(0, 0, 0, 0);
            if (p + r < p1) x = *reinterpret_cast<const uint4 *>(big + (size_t)(p + r) * width + a0 + cv * 8);
            *reinterpret_cast<uint4 *>(&big_s[r][cv * 8]) = x;
        }
        // small tile: 32 rows x R cols
        for (int v = tid; v < WG_P * R / 8; v += 128) {
            int r = v / (R / 8), cv = v % (R / 8);
            uint4 x = make_uint4(0, 0, 0, 0);
            if (p + r < p1) x = *reinterpret_cast<const uint4 *>(small_ + (size_t)(p + r) * kLoraPad + cv * 8);
            *reinterpret_cast<uint4 *>(&sm_s[r][cv * 8]) = x;
        }
        __syncthreads();
#pragma unroll
        for (int pp = 0; pp < WG_P; pp += 16) {
            wmma::fragment<wmma::matrix_b, 16, 16, 16, bf16, wmma::row_major> bfm;   // big[p][a]
            wmma::load_matrix_sync(bfm, &big_s[pp][warp * 16], WG_A + 8);
#pragma unroll
            for (int n = 0; n < R / 16; ++n) {
                wmma::fragment<wmma::matrix_a, 16, 16, 16, bf16, wmma::col_major> af;  // small^T[q][p]
                wmma::load_matrix_sync(af, &sm_s[pp][n * 16], R + 8);
                wmma::mma_sync(acc[n], af, bfm, acc[n]);
            }
        }
        __syncthreads();
    }
    const int a = a0 + warp * 16;
#pragma unroll
    for (int n = 0; n < R / 16; ++n) {
        if (out_ar)   // grad[e][a][q], ld = R: element (q, a) at a*R + q
            wmma::store_matrix_sync(grad + ((size_t)e * width + a) * R + n * 16, acc[n], R, wmma::mem_col_major);
        else          // grad[e][q][a], ld = width
            wmma::store_matrix_sync(grad + ((size_t)e * R + n * 16) * width + a, acc[n], width, wmma::mem_row_major);
    }
}

// r = 8: CUDA cores; thread per (a, q)
__global__ void __launch_bounds__(256) lora_wgrad_small_kernel(const bf16 *__restrict__ big, int width, int R,
                                                               const bf16 *__restrict__ small_, const int32_t *__restrict__ offsets,
                                                               int out_ar, float *__restrict__ grad) {
    const int e = blockIdx.x;
    const int p0 = offsets[e], p1 = offsets[e + 1];
    for (int v = blockIdx.y * 256 + threadIdx.x; v < width * R; v += gridDim.y * 256) {
        int a = v % width, q = v / width;
        float acc = 0.f;
        for (int p = p0; p < p1; ++p)
            acc = fmaf(__bfloat162float(small_[(size_t)p * kLoraPad + q]), __bfloat162float(big[(size_t)p * width + a]), acc);
        if (out_ar) grad[((size_t)e * width + a) * R + q] = acc;
        else grad[((size_t)e * R + q) * width + a] = acc;
    }
}

tqp_status launch_lora_wgrad(tqp_ctx *c, const bf16 *big, int width, const bf16 *small_, const int32_t *offsets,
                             int out_ar, float *grad, cudaStream_t st) {
    const int r = c->desc.r, E = c->desc.E;
    if (r == 16) lora_wgrad_kernel<16><<<dim3(E, width / WG_A), 128, 0, st>>>(big, width, small_, offsets, out_ar, grad);
    else if (r == 32) lora_wgrad_kernel<32><<<dim3(E, width / WG_A), 128, 0, st>>>(big, width, small_, offsets, out_ar, grad);
    else lora_wgrad_small_kernel<<<dim3(E, 8), 256, 0, st>>>(big, width, r, small_, offsets, out_ar, grad);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
