// Grouped dequant GEMM on the 5th-gen tensor cores (tcgen05 + TMEM + TMA), sm_100a.
//
//   out[p][m] = sum_seg sum_k act_seg[p][k] * W_seg[m][k]  +  sum_l lact_l[p][q] * lw_l[m][q]
//   W_seg[m][k] = bf16( bf16(codebook[code]) * bf16(scale) )       (look up, rescale by the norm)
//
// "Swap-AB": the UMMA M axis (always 128, always full) carries the weight output channels, the N axis carries
// the routed rows of ONE expert (16..256, multiples of 16), so ragged expert sizes cost <= 15 padded rows
// instead of a half-empty 128-row M tile.  The weight operand never exists in HBM as bf16: a TMA load brings the
// uint8 codes, four producer warps gather 16-byte codebook rows from a bank-conflict-free replicated LUT in
// shared memory, apply the per-channel scale and write the 128B-swizzled UMMA operand tile; the activation
// operand and the adapter projections arrive by TMA.  The rank-r adapter term is one extra K-step into the same
// TMEM accumulator.  Forward GEMMs contract along the code vectors (K-major A operand), backward GEMMs across
// them (MN-major A operand built from the same codes).
//
// Warp roles (320 threads, 1 CTA/SM, persistent over work items):  warp 0 TMA producer, warp 1 MMA issuer
// (+TMEM alloc), warps 2-5 dequant producers, warps 6-9 epilogue (TMEM -> registers -> bf16 -> global).
#include "common.cuh"

namespace tqp {
namespace g5 {

constexpr int BM = 128, BK = 64, TN = kTileRows;
constexpr int NSTAGE = 3, IDXQ = 3;
constexpr int X_BYTES = TN * 128, A_BYTES = BM * 128, IDX_BYTES = 128 * 16, LUT_BYTES = 256 * 8 * 16;
constexpr int OFF_X = 0, OFF_A = OFF_X + NSTAGE * X_BYTES, OFF_LUT = OFF_A + NSTAGE * A_BYTES,
              OFF_IDX = OFF_LUT + LUT_BYTES, OFF_BAR = OFF_IDX + IDXQ * IDX_BYTES;
constexpr int SMEM_BYTES = OFF_BAR + 256 + 1024;   // + alignment slack
constexpr int NTHREADS = 320;

// ---- PTX wrappers ----------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// one lane of a converged warp (ptxas then keeps the tcgen05.mma operands in uniform registers; see tc_ptx.cuh)
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done = 0;
    long long t0 = clock64();
    while (true) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
        if (done) break;
        if (clock64() - t0 > 8000000000ll) __trap();   // a broken pipeline must fault, not hang the GPU
    }
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void *tmap, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
        "l"(tmap), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum)
        : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t *v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// UMMA shared-memory descriptor (cute::UMMA::SmemDescriptor bit layout), SWIZZLE_128B, version 1
__device__ __forceinline__ uint64_t make_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((addr >> 4) & 0x3fff);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32;
    d |= (uint64_t)1 << 46;   // version = 1 (Blackwell)
    d |= (uint64_t)2 << 61;   // layout_type = SWIZZLE_128B
    return d;
}
// Instruction descriptor, kind::f16: D fp32, A/B bf16, M = 128, N = n; a_mn = 1 -> A is MN-major
__device__ __forceinline__ uint32_t make_idesc(int n, int a_mn) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | (0u << 16) | ((uint32_t)(n >> 3) << 17) |
           ((uint32_t)(BM >> 4) << 24);
}

struct Pipe {   // ring position + phase bit
    int s = 0;
    uint32_t ph = 0;
    __device__ __forceinline__ void next(int n) {
        if (++s == n) { s = 0; ph ^= 1; }
    }
};


// ---- the kernel ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NTHREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ GemmArgs args, const uint4 *__restrict__ lut_g, const Tile *__restrict__ tiles,
                    const int32_t *__restrict__ num_tiles_p, int ablate) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar0 = sbase + OFF_BAR;
    // barrier slots (8 bytes each)
    auto full_x = [&](int s) { return bar0 + 8u * s; };
    auto full_a = [&](int s) { return bar0 + 8u * (NSTAGE + s); };
    auto empty = [&](int s) { return bar0 + 8u * (2 * NSTAGE + s); };
    auto idx_full = [&](int s) { return bar0 + 8u * (3 * NSTAGE + s); };
    auto idx_empty = [&](int s) { return bar0 + 8u * (3 * NSTAGE + IDXQ + s); };
    auto tmem_full = [&](int s) { return bar0 + 8u * (3 * NSTAGE + 2 * IDXQ + s); };
    auto tmem_empty = [&](int s) { return bar0 + 8u * (3 * NSTAGE + 2 * IDXQ + 2 + s); };
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + OFF_BAR + 8 * (3 * NSTAGE + 2 * IDXQ + 4));

    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) { mbar_init(full_x(s), 1); mbar_init(full_a(s), 4); mbar_init(empty(s), 1); }
        for (int s = 0; s < IDXQ; ++s) { mbar_init(idx_full(s), 1); mbar_init(idx_empty(s), 4); }
        for (int s = 0; s < 2; ++s) { mbar_init(tmem_full(s), 1); mbar_init(tmem_empty(s), 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {   // TMEM: all 512 columns (two 256-column accumulators)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    {   // replicated LUT: entry e, copy c at (e*8 + c) * 16 B  ->  lane c of every quarter-warp hits bank group c
        uint4 *lut_s = reinterpret_cast<uint4 *>(smem + OFF_LUT);
        for (int i = threadIdx.x; i < 256 * 8; i += NTHREADS) lut_s[i] = lut_g[i >> 3];
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int num_tiles = *num_tiles_p;
    const int nprob = args.nprob;
    const int MT = args.p[0].M / BM;
    const long long total = (long long)num_tiles * nprob * MT;

    if (warp == 0) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            Pipe st, iq;
            for (long long item = blockIdx.x; item < total; item += gridDim.x) {
                const int tile_id = (int)(item / (nprob * MT)), rem = (int)(item % (nprob * MT));
                const Tile t = tiles[tile_id];
                if (t.rows <= 0) continue;
                const GemmProblem &pb = args.p[rem / MT];
                const int m0 = (rem % MT) * BM, M = pb.M;
                for (int sg = 0; sg < pb.nseg; ++sg) {
                    const GemmSeg &S = pb.seg[sg];
                    const int nkb = S.K / BK;
                    for (int kb = 0; kb < nkb; ++kb) {
                        if ((kb & 1) == 0) {
                            mbar_wait(idx_empty(iq.s), iq.ph ^ 1);
                            mbar_expect_tx(idx_full(iq.s), IDX_BYTES);
                            const int c0 = S.kmajor ? (kb >> 1) * 16 : m0 / 8;
                            const int c1 = S.kmajor ? t.expert * M + m0 : t.expert * S.K + kb * BK;
                            tma_load_2d(sbase + OFF_IDX + iq.s * IDX_BYTES, &S.idx_map, c0, c1, idx_full(iq.s));
                            iq.next(IDXQ);
                        }
                        mbar_wait(empty(st.s), st.ph ^ 1);
                        mbar_expect_tx(full_x(st.s), X_BYTES);
                        tma_load_2d(sbase + OFF_X + st.s * X_BYTES, &S.act_map, kb * BK, t.row0, full_x(st.s));
                        st.next(NSTAGE);
                    }
                }
                for (int l = 0; l < pb.nlora; ++l) {
                    mbar_wait(empty(st.s), st.ph ^ 1);
                    mbar_expect_tx(full_x(st.s), X_BYTES);
                    tma_load_2d(sbase + OFF_X + st.s * X_BYTES, &pb.lora[l].lact_map, 0, t.row0, full_x(st.s));
                    st.next(NSTAGE);
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        if (elect_one()) {
            Pipe st;
            int it = 0;
            for (long long item = blockIdx.x; item < total; item += gridDim.x) {
                const int tile_id = (int)(item / (nprob * MT)), rem = (int)(item % (nprob * MT));
                const Tile t = tiles[tile_id];
                if (t.rows <= 0) continue;
                const GemmProblem &pb = args.p[rem / MT];
                const int ab = it & 1;
                const uint32_t aph = (it >> 1) & 1;
                ++it;
                const int n = max(16, (t.rows + 15) & ~15);
                mbar_wait(tmem_empty(ab), aph ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + ab * TN;
                uint32_t accum = 0;
                for (int sg = 0; sg < pb.nseg; ++sg) {
                    const GemmSeg &S = pb.seg[sg];
                    const int nkb = S.K / BK;
                    const uint32_t idesc = make_idesc(n, S.kmajor ? 0 : 1);
                    for (int kb = 0; kb < nkb; ++kb) {
                        mbar_wait(full_x(st.s), st.ph);
                        mbar_wait(full_a(st.s), st.ph);
                        tc_fence_after();
                        const uint32_t xa = sbase + OFF_X + st.s * X_BYTES, aa = sbase + OFF_A + st.s * A_BYTES;
#pragma unroll
                        for (int kk = 0; kk < BK / 16; ++kk) {
                            const uint64_t bd = make_desc(xa + kk * 32, 16, 1024);
                            const uint64_t ad = S.kmajor ? make_desc(aa + kk * 32, 16, 1024) : make_desc(aa + kk * 4096, 1024, 2048);
                            umma_bf16(d_tmem, ad, bd, idesc, accum);
                            accum = 1;
                        }
                        umma_commit(empty(st.s));
                        st.next(NSTAGE);
                    }
                }
                const uint32_t idesc_l = make_idesc(n, 0);
                const int nmma_l = max(1, pb.r / 16);
                for (int l = 0; l < pb.nlora; ++l) {
                    mbar_wait(full_x(st.s), st.ph);
                    mbar_wait(full_a(st.s), st.ph);
                    tc_fence_after();
                    const uint32_t xa = sbase + OFF_X + st.s * X_BYTES, aa = sbase + OFF_A + st.s * A_BYTES;
                    for (int kk = 0; kk < nmma_l; ++kk) {
                        umma_bf16(d_tmem, make_desc(aa + kk * 32, 16, 1024), make_desc(xa + kk * 32, 16, 1024), idesc_l, accum);
                        accum = 1;
                    }
                    umma_commit(empty(st.s));
                    st.next(NSTAGE);
                }
                umma_commit(tmem_full(ab));
            }
        }
    } else if (warp < 6) {
        // =========================== dequant producers (128 threads) ===========================
        const int tid = threadIdx.x - 64;
        const int c = tid & 7;
        const uint4 *lut_s = reinterpret_cast<const uint4 *>(smem + OFF_LUT);
        Pipe st, iq;
        for (long long item = blockIdx.x; item < total; item += gridDim.x) {
            const int tile_id = (int)(item / (nprob * MT)), rem = (int)(item % (nprob * MT));
            const Tile t = tiles[tile_id];
            if (t.rows <= 0) continue;
            const GemmProblem &pb = args.p[rem / MT];
            const int m0 = (rem % MT) * BM, M = pb.M, e = t.expert;
            for (int sg = 0; sg < pb.nseg; ++sg) {
                const GemmSeg &S = pb.seg[sg];
                const int nkb = S.K / BK;
                const int kmajor = S.kmajor;
                // K-major: one scale per thread row for the whole tile.  MN-major: one per k-row per k-block.
                const __half *scale_p = S.scale + (kmajor ? (size_t)e * M + m0 + tid : (size_t)e * S.K + (tid & 63));
                __nv_bfloat162 s2 = __float2bfloat162_rn(__half2float(*scale_p));
                uint32_t codes[4];
                for (int kb = 0; kb < nkb; ++kb) {
                    if ((kb & 1) == 0) {
                        mbar_wait(idx_full(iq.s), iq.ph);
                        const uint8_t *is = smem + OFF_IDX + iq.s * IDX_BYTES;
                        if (kmajor) {
                            uint4 v = *reinterpret_cast<const uint4 *>(is + tid * 16);
                            codes[0] = v.x; codes[1] = v.y; codes[2] = v.z; codes[3] = v.w;
                        } else {
                            const int kr = tid & 63, half = tid >> 6;
                            uint2 v0 = *reinterpret_cast<const uint2 *>(is + kr * 16 + half * 8);
                            uint2 v1 = *reinterpret_cast<const uint2 *>(is + (64 + kr) * 16 + half * 8);
                            codes[0] = v0.x; codes[1] = v0.y; codes[2] = v1.x; codes[3] = v1.y;
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(idx_empty(iq.s));
                        iq.next(IDXQ);
                    }
                    if (!kmajor) s2 = __float2bfloat162_rn(__half2float(scale_p[kb * BK]));
                    const uint32_t c01[2] = {codes[(kb & 1) * 2], codes[(kb & 1) * 2 + 1]};
                    mbar_wait(empty(st.s), st.ph ^ 1);
                    uint8_t *as = smem + OFF_A + st.s * A_BYTES;
                    uint32_t rowoff, sw;
                    if (kmajor) { rowoff = tid * 128; sw = tid & 7; }
                    else {
                        const int kr = tid & 63, half = tid >> 6;
                        rowoff = ((kr >> 3) * 2 + half) * 1024 + (kr & 7) * 128;
                        sw = kr & 7;
                    }
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const uint32_t code = (c01[j >> 2] >> ((j & 3) * 8)) & 0xffu;
                        uint4 v = TQP_DBG(ablate & 1) ? make_uint4(code, code, code, code) : lut_s[code * 8 + c];
                        __nv_bfloat162 *pv = reinterpret_cast<__nv_bfloat162 *>(&v);
                        if (!TQP_DBG(ablate & 4)) {
#pragma unroll
                            for (int q = 0; q < 4; ++q) pv[q] = __hmul2(pv[q], s2);
                        }
                        if (!TQP_DBG(ablate & 2)) *reinterpret_cast<uint4 *>(as + rowoff + ((j ^ sw) << 4)) = v;
                    }
                    fence_async_smem();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(full_a(st.s));
                    st.next(NSTAGE);
                }
            }
            // adapter K-step: A tile = lw[m0 + tid][0..r) as a K-major row (chunks beyond r zeroed)
            const int r = pb.r, nch = 2 * max(1, r / 16);
            for (int l = 0; l < pb.nlora; ++l) {
                const GemmLora &L = pb.lora[l];
                uint4 ch[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) ch[j] = make_uint4(0, 0, 0, 0);
                if (L.mk_layout) {
                    const uint4 *src = reinterpret_cast<const uint4 *>(L.lw + ((size_t)e * M + m0 + tid) * r);
                    for (int j = 0; j < r / 8; ++j) ch[j] = src[j];
                } else {
                    const bf16 *src = L.lw + (size_t)e * r * M + m0 + tid;
                    uint16_t *h = reinterpret_cast<uint16_t *>(ch);
                    for (int q = 0; q < r; ++q) h[q] = *reinterpret_cast<const uint16_t *>(src + (size_t)q * M);
                }
                mbar_wait(empty(st.s), st.ph ^ 1);
                uint8_t *as = smem + OFF_A + st.s * A_BYTES;
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (j < nch) *reinterpret_cast<uint4 *>(as + tid * 128 + ((j ^ (tid & 7)) << 4)) = ch[j];
                fence_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(full_a(st.s));
                st.next(NSTAGE);
            }
        }
    } else {
        // =========================== epilogue (128 threads) ===========================
        const int q = warp & 3;             // TMEM lane quadrant this warp may access
        const int m = q * 32 + lane;        // output channel inside the tile
        int it = 0;
        for (long long item = blockIdx.x; item < total; item += gridDim.x) {
            const int tile_id = (int)(item / (nprob * MT)), rem = (int)(item % (nprob * MT));
            const Tile t = tiles[tile_id];
            if (t.rows <= 0) continue;
            const GemmProblem &pb = args.p[rem / MT];
            const int m0 = (rem % MT) * BM, M = pb.M;
            const int ab = it & 1;
            const uint32_t aph = (it >> 1) & 1;
            ++it;
            mbar_wait(tmem_full(ab), aph);
            tc_fence_after();
            bf16 *outp = pb.out + (size_t)t.row0 * M + m0 + m;
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + ab * TN;
            for (int c0 = 0; c0 < t.rows; c0 += 16) {
                uint32_t v[16];
                tmem_ld16(taddr + c0, v);
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 16; ++j)
                    if (c0 + j < t.rows) outp[(size_t)(c0 + j) * M] = __float2bfloat16_rn(__uint_as_float(v[j]));
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tmem_empty(ab));
        }
    }

    __syncwarp();
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512));
    }
}

}  // namespace g5

tqp_status launch_gemm_tcgen05(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st) {
    if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&g5::gemm_tcgen05_kernel), g5::SMEM_BYTES)) return st_attr;
    GemmArgs args;
    for (int i = 0; i < nprob; ++i) args.p[i] = probs[i];
    args.nprob = nprob;
    g5::gemm_tcgen05_kernel<<<c->num_sms, g5::NTHREADS, g5::SMEM_BYTES, st>>>(
        args, c->p<uint4>(c->ws.lut), c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles), c->ablate);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
