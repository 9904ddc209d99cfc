// Consolidation (§10.6): the trained adapter is merged into the dequantised base and the result
// is materialised as bf16,  W[e][out][in] = bf16( scale[out] * codebook[idx[out][in/8]][in%8] + s * sum_q A[in][q] B[q][out] ),
// one row per output channel (the layout of the code indices; "ordinary weights" for a dense y = x W^T).
// fp32 accumulation, one rounding at the end.  Bound: HBM writes (2 bytes per weight; 7.2 GB for the three packs of
// cfg 2); a release step, not part of the timed layer.
//
// r = 16 / 32: the adapter product is a dense rank-r contraction and runs on the tensor cores (mma.sync.m16n8k16, one or
// two k-steps): M = 16 output channels (operand s.t. (m, k) = B[k][m], from a shared-memory tile by ldmatrix.trans),
// N = 8 input columns (operand (k, n) = A[n][k]: the rows of A as they lie in memory, one 8-byte load per thread with
// the k slots permuted so that a thread's two k-pairs are adjacent: slot 2t+e <-> rank 4t+e, slot 8+2t+e <-> rank
// 4t+2+e; the other operand's ldmatrix rows are picked to match).  The accumulator gives a thread 2 columns of 16
// n-blocks; a 4x4 transpose inside each quad (two xor-shuffle stages) turns that into 8 consecutive columns of one
// n-block = one code vector, so the base value is one 16-byte codebook load and the store is 16 bytes per thread.
// r = 8 (config 0): CUDA-core kernel below (r FMAs per weight).
#include "common.cuh"

namespace tqp {

__device__ __forceinline__ void cs_ldsm_x4_t(uint32_t addr, uint32_t (&r)[4]) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void cs_mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// 4x4 transpose of x[0..3] across the four lanes of a quad: afterwards x[s] is what lane s of the quad held in x[t]
__device__ __forceinline__ void quad_transpose(float (&x)[4], int t) {
    const bool o1 = t & 1, o2 = t & 2;
    float s0 = o1 ? x[0] : x[1], s1 = o1 ? x[2] : x[3];
    s0 = __shfl_xor_sync(0xffffffffu, s0, 1);
    s1 = __shfl_xor_sync(0xffffffffu, s1, 1);
    if (o1) { x[0] = s0; x[2] = s1; } else { x[1] = s0; x[3] = s1; }
    s0 = o2 ? x[0] : x[2];
    s1 = o2 ? x[1] : x[3];
    s0 = __shfl_xor_sync(0xffffffffu, s0, 2);
    s1 = __shfl_xor_sync(0xffffffffu, s1, 2);
    if (o2) { x[0] = s0; x[1] = s1; } else { x[2] = s0; x[3] = s1; }
}

constexpr int CM_IN = 128, CM_OUT = 128, CM_BLD = CM_OUT + 8;   // CTA tile; padded row of the B tile

// grid (in / 128, out / 128, experts), 256 threads: warp w owns output channels o0 + 16 w .. + 16, all 128 input columns
template <int R>
__global__ void __launch_bounds__(256) consolidate_mma_kernel(const uint8_t *__restrict__ idx, const __half *__restrict__ scale,
                                                              const __half *__restrict__ codebook, const bf16 *__restrict__ A,
                                                              const bf16 *__restrict__ B, int in_dim, int out_dim, float s, int e0,
                                                              bf16 *__restrict__ W) {
    __shared__ __align__(16) bf16 b_s[R][CM_BLD];   // B[e][q][o0 ..]
    const int e = e0 + blockIdx.z, i0 = blockIdx.x * CM_IN, o0 = blockIdx.y * CM_OUT;
    const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32, g = lane / 4, t = lane % 4;
    for (int v = tid; v < R * (CM_OUT / 8); v += 256) {
        const int q = v / (CM_OUT / 8), c8 = (v % (CM_OUT / 8)) * 8;
        *reinterpret_cast<uint4 *>(&b_s[q][c8]) = *reinterpret_cast<const uint4 *>(B + ((size_t)e * R + q) * out_dim + o0 + c8);
    }
    __syncthreads();
    float acc[CM_IN / 8][4];
#pragma unroll
    for (int nb = 0; nb < CM_IN / 8; ++nb)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[nb][c] = 0.f;
    const int li = lane % 8, mat = lane / 8;
    const bf16 *arow = A + ((size_t)e * in_dim + i0 + g) * R + 4 * t;   // this thread's 4 adjacent ranks of row i0 + 8 nb + g
#pragma unroll
    for (int ks = 0; ks < R / 16; ++ks) {
        uint32_t af[4];
        const int q = 16 * ks + 4 * (li / 2) + (li % 2) + 2 * (mat / 2);
        cs_ldsm_x4_t((uint32_t)__cvta_generic_to_shared(&b_s[q][warp * 16 + 8 * (mat % 2)]), af);
#pragma unroll
        for (int nb = 0; nb < CM_IN / 8; ++nb) {
            const uint2 bv = __ldg(reinterpret_cast<const uint2 *>(arow + (size_t)nb * 8 * R + 16 * ks));
            cs_mma16816(acc[nb], af, bv.x, bv.y);
        }
    }
    const int nvec = in_dim / 8;
#pragma unroll
    for (int h = 0; h < 2; ++h) {   // rows g and g + 8 of the warp's 16
        const int o = o0 + warp * 16 + g + 8 * h;
        const float sc = __half2float(scale[(size_t)e * out_dim + o]);
        const uint8_t *irow = idx + ((size_t)e * out_dim + o) * nvec + i0 / 8;
        bf16 *wrow = W + ((size_t)blockIdx.z * out_dim + o) * in_dim + i0;
#pragma unroll
        for (int grp = 0; grp < CM_IN / 32; ++grp) {   // four n-blocks at a time: after the transposes lane t holds n-block 4 grp + t
            float lo[4], hi[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) { lo[j] = acc[4 * grp + j][2 * h]; hi[j] = acc[4 * grp + j][2 * h + 1]; }
            quad_transpose(lo, t);
            quad_transpose(hi, t);   // columns 2 s, 2 s + 1 of the block are lo[s], hi[s]
            const int nb = 4 * grp + t;
            const uint4 cv = __ldg(reinterpret_cast<const uint4 *>(codebook) + irow[nb]);
            const __half2 *ch = reinterpret_cast<const __half2 *>(&cv);
            uint4 ov;
            uint32_t *op = reinterpret_cast<uint32_t *>(&ov);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float2 f = __half22float2(ch[j]);
                op[j] = float2_to_bf16x2(fmaf(s, lo[j], sc * f.x), fmaf(s, hi[j], sc * f.y));
            }
            *reinterpret_cast<uint4 *>(wrow + nb * 8) = ov;
        }
    }
}

constexpr int CS_IN = 256;    // input columns per CTA: 32 lanes x one 8-vector
constexpr int CS_OUT = 64;    // output rows per CTA: 8 warps x 8
constexpr int CS_RMAX = 32;

// A [E][in][r] bf16, B [E][r][out] bf16, idx [E][out][in/8], scale fp16 [E][out], codebook fp16 [256][8]
__global__ void __launch_bounds__(256) consolidate_kernel(const uint8_t *__restrict__ idx, const __half *__restrict__ scale,
                                                          const __half *__restrict__ codebook, const bf16 *__restrict__ A,
                                                          const bf16 *__restrict__ B, int in_dim, int out_dim, int r, float s, int e0,
                                                          bf16 *__restrict__ W) {
    __shared__ float a_s[CS_RMAX][8][33];   // A[i0 + 8 lane + j][q] at [q][j][lane]: lanes read consecutive words
    __shared__ float b_s[CS_RMAX][CS_OUT];  // s * B[q][o0 + o]
    const int e = e0 + blockIdx.z, i0 = blockIdx.x * CS_IN, o0 = blockIdx.y * CS_OUT;
    const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
    for (int v = tid; v < CS_IN * r / 8; v += 256) {   // 16 bytes = 8 ranks of one row of A
        const int i = v / (r / 8), q0 = (v % (r / 8)) * 8;
        uint4 av = make_uint4(0, 0, 0, 0);
        if (i0 + i < in_dim) av = *reinterpret_cast<const uint4 *>(A + ((size_t)e * in_dim + i0 + i) * r + q0);
        const uint32_t *ap = reinterpret_cast<const uint32_t *>(&av);
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const float2 f = bf16x2_to_float2(ap[h]);
            a_s[q0 + 2 * h][i % 8][i / 8] = f.x;
            a_s[q0 + 2 * h + 1][i % 8][i / 8] = f.y;
        }
    }
    for (int v = tid; v < r * CS_OUT; v += 256) {
        const int q = v / CS_OUT, o = v % CS_OUT;
        b_s[q][o] = o0 + o < out_dim ? s * __bfloat162float(B[((size_t)e * r + q) * out_dim + o0 + o]) : 0.f;
    }
    __syncthreads();
    const int ic = i0 + 8 * lane;   // this lane's 8 input columns
    if (ic >= in_dim) return;
    const int nvec = in_dim / 8;
    constexpr int NR = CS_OUT / 8;   // output rows per warp
    float acc[NR][8];                // s (A B)[ic + j][o] of this lane's 8 columns and this warp's rows
#pragma unroll
    for (int oo = 0; oo < NR; ++oo)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[oo][j] = 0.f;
    for (int q = 0; q < r; ++q) {    // 16 shared-memory loads per 64 FMAs
        float av[8], bv[NR];
#pragma unroll
        for (int j = 0; j < 8; ++j) av[j] = a_s[q][j][lane];
#pragma unroll
        for (int oo = 0; oo < NR; ++oo) bv[oo] = b_s[q][warp * NR + oo];
#pragma unroll
        for (int oo = 0; oo < NR; ++oo)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[oo][j] = fmaf(av[j], bv[oo], acc[oo][j]);
    }
#pragma unroll
    for (int oo = 0; oo < NR; ++oo) {
        const int o = o0 + warp * NR + oo;
        if (o >= out_dim) break;
        const int code = idx[((size_t)e * out_dim + o) * nvec + ic / 8];
        const float sc = __half2float(scale[(size_t)e * out_dim + o]);
        const uint4 cv = __ldg(reinterpret_cast<const uint4 *>(codebook) + code);   // 4 KB table: L1-resident
        const __half2 *ch = reinterpret_cast<const __half2 *>(&cv);
        uint4 ov;
        uint32_t *op = reinterpret_cast<uint32_t *>(&ov);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float2 f = __half22float2(ch[j]);
            op[j] = float2_to_bf16x2(fmaf(sc, f.x, acc[oo][2 * j]), fmaf(sc, f.y, acc[oo][2 * j + 1]));
        }
        *reinterpret_cast<uint4 *>(W + ((size_t)blockIdx.z * out_dim + o) * in_dim + ic) = ov;
    }
}

tqp_status launch_consolidate(tqp_ctx *c, int pack, int e0, int n_experts, bf16 *W, cudaStream_t st) {
    const tqp_layer_desc &D = c->desc;
    const bool down = pack == 2;
    const int in_dim = down ? D.F : D.d, out_dim = down ? D.d : D.F;
    const uint8_t *idx = pack == 0 ? c->w.idx_gate : pack == 1 ? c->w.idx_up : c->w.idx_down;
    const void *scale = pack == 0 ? c->w.scale_gate : pack == 1 ? c->w.scale_up : c->w.scale_down;
    const void *A = pack == 0 ? c->w.A_gate : pack == 1 ? c->w.A_up : c->w.A_down;
    const void *B = pack == 0 ? c->w.B_gate : pack == 1 ? c->w.B_up : c->w.B_down;
    for (int z0 = 0; z0 < n_experts; z0 += 32768) {   // gridDim.z limit
        const int nz = std::min(32768, n_experts - z0);
        if (D.r == 16 || D.r == 32) {   // in, out % 128 == 0 by the layer's constraints
            dim3 gm(in_dim / CM_IN, out_dim / CM_OUT, nz);
            bf16 *wz = W + (size_t)z0 * out_dim * in_dim;
            if (D.r == 16)
                consolidate_mma_kernel<16><<<gm, 256, 0, st>>>(idx, (const __half *)scale, (const __half *)c->w.codebook, (const bf16 *)A,
                                                               (const bf16 *)B, in_dim, out_dim, D.lora_scale, e0 + z0, wz);
            else
                consolidate_mma_kernel<32><<<gm, 256, 0, st>>>(idx, (const __half *)scale, (const __half *)c->w.codebook, (const bf16 *)A,
                                                               (const bf16 *)B, in_dim, out_dim, D.lora_scale, e0 + z0, wz);
            TQP_LAUNCH_OK(c);
            continue;
        }
        dim3 grid((in_dim + CS_IN - 1) / CS_IN, (out_dim + CS_OUT - 1) / CS_OUT, nz);
        consolidate_kernel<<<grid, 256, 0, st>>>(idx, (const __half *)scale, (const __half *)c->w.codebook, (const bf16 *)A, (const bf16 *)B,
                                                 in_dim, out_dim, D.r, D.lora_scale, e0 + z0, W + (size_t)z0 * out_dim * in_dim);
        TQP_LAUNCH_OK(c);
    }
    return TQP_OK;
}

}  // namespace tqp
