// CUDA-core scaffold of the grouped dequant GEMM (debug / ablation reference for gemm_tcgen05.cu; selected with
// tqp_set_option("gemm_impl", 1)).  Same contract and the same operand rounding as the tensor-core kernel:
//   out[p][m] = sum_seg sum_k act[p][k] * bf16(bf16(cb[code]) * bf16(scale)) + sum_l lact[p][q] * lw[m][q]
// with fp32 accumulation.  Slow on purpose: obviously-correct smem tiling, no tensor cores.
#include "common.cuh"

namespace tqp {

constexpr int SC_M = 64, SC_K = 64, SC_R = 32;

__device__ __forceinline__ float deq_elem(const GemmSeg &sg, const bf16 *lut, int e, int M, int m, int kx) {
    // kmajor: idx[e][M][K/8], scale[e][M];  else idx[e][K][M/8], scale[e][K]
    int code;
    float sc;
    if (sg.kmajor) {
        code = sg.idx[((size_t)e * M + m) * (sg.K / 8) + kx / 8];
        sc = __bfloat162float(__float2bfloat16_rn(__half2float(sg.scale[(size_t)e * M + m])));
        return __bfloat162float(__float2bfloat16_rn(__bfloat162float(lut[code * 8 + kx % 8]) * sc));
    }
    code = sg.idx[((size_t)e * sg.K + kx) * (M / 8) + m / 8];
    sc = __bfloat162float(__float2bfloat16_rn(__half2float(sg.scale[(size_t)e * sg.K + kx])));
    return __bfloat162float(__float2bfloat16_rn(__bfloat162float(lut[code * 8 + m % 8]) * sc));
}

// grid = (max_tiles, M/64, nprob), block = 256: thread (r = tid/8, mg = tid%8) owns rows {sb*32 + r} x columns {mg + 8j}
__global__ void __launch_bounds__(256) gemm_scaffold_kernel(const __grid_constant__ GemmArgs args, const bf16 *__restrict__ lut,
                                                            const Tile *__restrict__ tiles, const int32_t *__restrict__ num_tiles) {
    __shared__ float W_s[SC_K][SC_M + 1];
    __shared__ float A_s[SC_R][SC_K + 1];
    if ((int)blockIdx.x >= *num_tiles) return;
    const Tile t = tiles[blockIdx.x];
    if (t.rows <= 0) return;
    const GemmProblem &pb = args.p[blockIdx.z];
    const int M = pb.M, m0 = blockIdx.y * SC_M, tid = threadIdx.x, r = tid / 8, mg = tid % 8, e = t.expert;
    float acc[kTileRows / SC_R][8];
#pragma unroll
    for (int sb = 0; sb < kTileRows / SC_R; ++sb)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[sb][j] = 0.f;

    const int nsteps_lora = pb.nlora;
    for (int part = 0; part < pb.nseg + nsteps_lora; ++part) {
        const bool is_lora = part >= pb.nseg;
        const int K = is_lora ? pb.r : pb.seg[part].K;
        const bf16 *act = is_lora ? pb.lora[part - pb.nseg].lact : pb.seg[part].act;
        const int lda = is_lora ? kLoraPad : K;
        for (int k0 = 0; k0 < K; k0 += SC_K) {
            const int kc = min(SC_K, K - k0);
            __syncthreads();
            for (int v = tid; v < SC_K * SC_M; v += 256) {
                int kk = v / SC_M, mm = v % SC_M;
                float w = 0.f;
                if (kk < kc) {
                    if (is_lora) {
                        const GemmLora &lr = pb.lora[part - pb.nseg];
                        w = __bfloat162float(lr.mk_layout ? lr.lw[((size_t)e * M + m0 + mm) * pb.r + k0 + kk]
                                                          : lr.lw[((size_t)e * pb.r + k0 + kk) * M + m0 + mm]);
                    } else {
                        w = deq_elem(pb.seg[part], lut, e, M, m0 + mm, k0 + kk);
                    }
                }
                W_s[kk][mm] = w;
            }
#pragma unroll 1
            for (int sb = 0; sb * SC_R < t.rows; ++sb) {
                __syncthreads();
                for (int v = tid; v < SC_R * SC_K; v += 256) {
                    int rr = v / SC_K, kk = v % SC_K;
                    int row = sb * SC_R + rr;
                    A_s[rr][kk] = (row < t.rows && kk < kc) ? __bfloat162float(act[(size_t)(t.row0 + row) * lda + k0 + kk]) : 0.f;
                }
                __syncthreads();
#pragma unroll 4
                for (int kk = 0; kk < SC_K; ++kk) {
                    float a = A_s[r][kk];
#pragma unroll
                    for (int j = 0; j < 8; ++j) acc[sb][j] = fmaf(a, W_s[kk][mg + 8 * j], acc[sb][j]);
                }
            }
        }
    }
#pragma unroll
    for (int sb = 0; sb < kTileRows / SC_R; ++sb) {
        int row = sb * SC_R + r;
        if (row < t.rows)
#pragma unroll
            for (int j = 0; j < 8; ++j) pb.out[(size_t)(t.row0 + row) * M + m0 + mg + 8 * j] = __float2bfloat16_rn(acc[sb][j]);
    }
}

tqp_status launch_gemm_scaffold(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st) {
    GemmArgs args;
    for (int i = 0; i < nprob; ++i) args.p[i] = probs[i];
    args.nprob = nprob;
    dim3 grid(c->max_tiles, probs[0].M / SC_M, nprob);
    gemm_scaffold_kernel<<<grid, 256, 0, st>>>(args, c->p<bf16>(c->ws.lut), c->p<Tile>(c->ws.tiles),
                                               c->p<int32_t>(c->ws.num_tiles));
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
