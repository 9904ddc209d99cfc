// Grouped dequant GEMM on CTA PAIRS (tcgen05 cta_group::2 + TMEM + TMA), sm_100a — the default GEMM of the layer.
//
//   out[p][m] = sum_seg sum_k act_seg[p][k] * W_seg[m][k]  +  sum_l lact_l[p][q] * lw_l[m][q]
//   W_seg[m][k] = bf16( bf16(codebook[code]) * bf16(scale) )       (look up, rescale by the norm)
//
// Same "swap-AB" mapping as gemm_tcgen05.cu (UMMA M = weight output channels, N = routed rows of one expert), but
// one UMMA instruction spans two SMs: M = 256 (each CTA dequantises and owns 128 output channels), and the routed
// rows (B operand) are split between the two CTAs' shared memories, so every SM loads, stores and re-reads only
// half of the activation tile.  That halves the shared-memory traffic of the activation operand, which — next to
// the codebook gathers — is what bounds this kernel.
//
// Warp roles per CTA (480 threads, 1 CTA/SM, persistent over work items, cluster = 2 CTAs):
//   warp 0  TMA producer of the activation / adapter-projection tiles (signals the LEADER's barrier)
//   warp 1  MMA issuer (leader CTA only) + TMEM allocation
//   warp 2  TMA producer of the code-index tiles (deep ring: indices stream from HBM exactly once)
//   warps 3-10  dequant producers, two groups of four that alternate K-blocks
//   warps 11-14 epilogue (TMEM -> registers -> bf16 -> global)
#include "common.cuh"
#include "tc_ptx.cuh"

namespace tqp {
namespace g2 {
using namespace ptx;

constexpr int BM = 128, BK = 64, TN = kTileRows, HN = kTileRows / 2;
constexpr int NSTAGE = 5, IDXQ = 8;
constexpr int X_BYTES = HN * 128, A_BYTES = BM * 128, IDX_BYTES = 128 * 16, LUT_BYTES = 256 * 8 * 16;
constexpr int OFF_X = 0, OFF_A = OFF_X + NSTAGE * X_BYTES, OFF_LUT = OFF_A + NSTAGE * A_BYTES,
              OFF_IDX = OFF_LUT + LUT_BYTES, OFF_BAR = OFF_IDX + IDXQ * IDX_BYTES, OFF_EPI = OFF_BAR + 512;
constexpr int EPI_ROWS = 32, EPI_BYTES = EPI_ROWS * BM * 2;   // output staging: [32 rows][128 channels] bf16, two buffers
constexpr int SMEM_BYTES = OFF_EPI + 2 * EPI_BYTES + 1024;
constexpr int NTHREADS = 480;
constexpr int W_DEQ0 = 3, W_EPI0 = 11;

struct Item {
    Tile t;
    int prob, m0;
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
gemm_tcgen05_2cta_kernel(const __grid_constant__ GemmArgs args, const uint4 *__restrict__ lut_g, const Tile *__restrict__ tiles,
                         const int32_t *__restrict__ num_tiles_p, int ablate, long long *__restrict__ trace) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar0 = sbase + OFF_BAR;
    // full[s] (the LEADER's is used): 1 arrival + 2 x X_BYTES of TMA from the activation producers, 8 dequant-warp arrivals
    auto full = [&](int s) { return bar0 + 8u * s; };
    auto empty = [&](int s) { return bar0 + 8u * (2 * NSTAGE + s); };                // local, multicast commit
    auto idx_full = [&](int s) { return bar0 + 8u * (3 * NSTAGE + s); };             // local
    auto idx_empty = [&](int s) { return bar0 + 8u * (3 * NSTAGE + IDXQ + s); };     // local
    auto tmem_full = [&](int s) { return bar0 + 8u * (3 * NSTAGE + 2 * IDXQ + s); }; // local, multicast commit
    auto tmem_empty = [&](int s) { return bar0 + 8u * (3 * NSTAGE + 2 * IDXQ + 2 + s); };   // leader's is used
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + OFF_BAR + 8 * (3 * NSTAGE + 2 * IDXQ + 4));

    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const uint32_t rank = cluster_ctarank();
    const uint32_t full_remote = mapa(full(0), 0), tmem_empty_remote = mapa(tmem_empty(0), 0);   // the leader's barriers

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) { mbar_init(full(s), 9); mbar_init(empty(s), 1); }
        for (int s = 0; s < IDXQ; ++s) { mbar_init(idx_full(s), 1); mbar_init(idx_empty(s), 8); }
        for (int s = 0; s < 2; ++s) { mbar_init(tmem_full(s), 1); mbar_init(tmem_empty(s), 8); }
        mbar_init_fence();
    }
    if (warp == 1) tmem_alloc<2>(smem_u32(tmem_slot), 512);
    {   // replicated LUT: entry e, copy c at (e*8 + c) * 16 B  ->  lane c of every quarter-warp hits bank group c
        uint4 *lut_s = reinterpret_cast<uint4 *>(smem + OFF_LUT);
        for (int i = threadIdx.x; i < 256 * 8; i += NTHREADS) lut_s[i] = lut_g[i >> 3];
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync();   // both CTAs' barriers are initialised before any remote arrive / TMA completion
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int num_tiles = *num_tiles_p;
    const int nprob = args.nprob;
    const int MTP = args.p[0].M / (2 * BM);
    const long long total = (long long)num_tiles * nprob * MTP;
    const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;

    auto get_item = [&](long long item, Item &it) {
        const int tile_id = (int)(item / (nprob * MTP)), rem = (int)(item % (nprob * MTP));
        it.t = tiles[tile_id];
        it.prob = rem / MTP;
        it.m0 = ((rem % MTP) * 2 + (int)rank) * BM;
    };

    if (warp == 0) {
        // =========================== activation TMA producer ===========================
        if (lane == 0) {
            Pipe st;
            for (long long item = cid; item < total; item += ncl) {
                Item it;
                get_item(item, it);
                if (it.t.rows <= 0) continue;
                const GemmProblem &pb = args.p[it.prob];
                const int n = max(16, (it.t.rows + 15) & ~15);
                const int row = it.t.row0 + (int)rank * (n >> 1);
                for (int sg = 0; sg < pb.nseg; ++sg) {
                    const GemmSeg &S = pb.seg[sg];
                    const int nkb = S.K / BK;
                    for (int kb = 0; kb < nkb; ++kb) {
                        mbar_wait(empty(st.s), st.ph ^ 1);
                        if (TQP_DBG(ablate & 8)) { if (rank == 0) mbar_arrive(full(st.s)); st.next(NSTAGE); continue; }
                        if (rank == 0) mbar_expect_tx(full(st.s), 2 * X_BYTES);
                        tma_load_2d_pair(sbase + OFF_X + st.s * X_BYTES, &S.act_map2, kb * BK, row, full_remote + 8u * st.s);
                        st.next(NSTAGE);
                    }
                }
                for (int l = 0; l < pb.nlora; ++l) {
                    mbar_wait(empty(st.s), st.ph ^ 1);
                    if (rank == 0) mbar_expect_tx(full(st.s), 2 * X_BYTES);
                    tma_load_2d_pair(sbase + OFF_X + st.s * X_BYTES, &pb.lora[l].lact_map2, 0, row, full_remote + 8u * st.s);
                    st.next(NSTAGE);
                }
            }
        }
    } else if (warp == 2) {
        // =========================== code-index TMA producer ===========================
        if (lane == 0) {
            Pipe iq;
            for (long long item = cid; item < total; item += ncl) {
                Item it;
                get_item(item, it);
                if (it.t.rows <= 0) continue;
                const GemmProblem &pb = args.p[it.prob];
                for (int sg = 0; sg < pb.nseg; ++sg) {
                    const GemmSeg &S = pb.seg[sg];
                    const int npair = S.K / (2 * BK);
                    for (int kp = 0; kp < npair; ++kp) {
                        mbar_wait(idx_empty(iq.s), iq.ph ^ 1);
                        if (TQP_DBG(ablate & 64)) { mbar_arrive(idx_full(iq.s)); iq.next(IDXQ); continue; }
                        mbar_expect_tx(idx_full(iq.s), IDX_BYTES);
                        const int c0 = S.kmajor ? kp * 16 : it.m0 / 8;
                        const int c1 = S.kmajor ? it.t.expert * pb.M + it.m0 : it.t.expert * S.K + kp * 2 * BK;
                        tma_load_2d(sbase + OFF_IDX + iq.s * IDX_BYTES, &S.idx_map, c0, c1, idx_full(iq.s));
                        iq.next(IDXQ);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer (leader CTA) ===========================
        if (rank == 0 && elect_one()) {
            Pipe st;
            int cnt = 0, tcount = 0;
            for (long long item = cid; item < total; item += ncl) {
                Item it;
                get_item(item, it);
                if (it.t.rows <= 0) continue;
                const GemmProblem &pb = args.p[it.prob];
                const int ab = cnt & 1;
                const uint32_t aph = (cnt >> 1) & 1;
                ++cnt;
                const int n = max(16, (it.t.rows + 15) & ~15);
                mbar_wait<true>(tmem_empty(ab), aph ^ 1);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + ab * TN;
                uint32_t accum = 0;
                const uint32_t hi_k = desc_hi(1024), lo_k = desc_lo_const(16);          // K-major SW128: SBO = 8 rows x 128 B
                const uint32_t hi_mn = desc_hi(2048), lo_mn = desc_lo_const(1024);      // MN-major SW128 A tile
                const uint32_t x16 = (sbase + OFF_X) >> 4, a16 = (sbase + OFF_A) >> 4;
                for (int sg = 0; sg < pb.nseg; ++sg) {
                    const GemmSeg &S = pb.seg[sg];
                    const int nkb = S.K / BK;
                    const int kmajor = S.kmajor;
                    const uint32_t idesc = make_idesc(2 * BM, n, kmajor ? 0 : 1);
                    const uint32_t a_hi = kmajor ? hi_k : hi_mn, a_lo = kmajor ? lo_k : lo_mn, a_step = kmajor ? 2u : 256u;
                    for (int kb = 0; kb < nkb; ++kb) {
                        long long tr0 = 0;
                        if (TQP_DBG(trace != nullptr) && cid == 0) tr0 = clock64();
                        mbar_wait<true>(full(st.s), st.ph);
                        tc_fence_after();
                        if (TQP_DBG(trace != nullptr) && cid == 0 && tcount < 2000) { trace[tcount * 4 + 0] = tr0; trace[tcount * 4 + 1] = clock64(); }
                        const uint32_t xs = x16 + st.s * (X_BYTES >> 4), as = a16 + st.s * (A_BYTES >> 4);
#pragma unroll
                        for (int kk = 0; kk < BK / 16; ++kk) {
                            if (TQP_DBG(ablate & 32)) break;
                            umma_bf16<2>(d_tmem, desc_from(a_hi, a_lo, as + kk * a_step), desc_from(hi_k, lo_k, xs + kk * 2), idesc, accum);
                            accum = 1;
                        }
                        umma_commit_pair(empty(st.s), 3);
                        if (TQP_DBG(trace != nullptr) && cid == 0 && tcount < 2000) { trace[tcount * 4 + 2] = clock64(); trace[tcount * 4 + 3] = kb; ++tcount; }
                        st.next(NSTAGE);
                    }
                }
                const uint32_t idesc_l = make_idesc(2 * BM, n, 0);
                const int nmma_l = max(1, pb.r / 16);
                for (int l = 0; l < pb.nlora; ++l) {
                    mbar_wait<true>(full(st.s), st.ph);
                    tc_fence_after();
                    const uint32_t xs = x16 + st.s * (X_BYTES >> 4), as = a16 + st.s * (A_BYTES >> 4);
                    for (int kk = 0; kk < nmma_l; ++kk) {
                        umma_bf16<2>(d_tmem, desc_from(hi_k, lo_k, as + kk * 2), desc_from(hi_k, lo_k, xs + kk * 2), idesc_l, accum);
                        accum = 1;
                    }
                    umma_commit_pair(empty(st.s), 3);
                    st.next(NSTAGE);
                }
                umma_commit_pair(tmem_full(ab), 3);
            }
        }
    } else if (warp >= W_DEQ0 && warp < W_EPI0) {
        // =========================== dequant producers: 2 groups x 128 threads ===========================
        const int g = (warp - W_DEQ0) >> 2;
        const int tid = (threadIdx.x - W_DEQ0 * 32) & 127;
        const int c = tid & 7;
        const uint32_t lut_a = sbase + OFF_LUT + c * 16;
        Pipe st, iq;
        int dcount = 0;
        for (long long item = cid; item < total; item += ncl) {
            Item it;
            get_item(item, it);
            if (it.t.rows <= 0) continue;
            const GemmProblem &pb = args.p[it.prob];
            const int m0 = it.m0, M = pb.M, e = it.t.expert;
            // adapter rows of this item's K-step(s): fetched now, consumed after the k-loop (latency hidden behind it)
            const int r = pb.r, nch = 2 * max(1, r / 16);
            uint4 ch[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) ch[j] = make_uint4(0, 0, 0, 0);
            for (int l = 0; l < pb.nlora; ++l) {
                if ((l & 1) == g) {   // at most one adapter step per group and item (nlora <= 2)
                    const GemmLora &L = pb.lora[l];
                    if (L.mk_layout) {
                        const uint4 *src = reinterpret_cast<const uint4 *>(L.lw + ((size_t)e * M + m0 + tid) * r);
                        for (int j = 0; j < r / 8; ++j) ch[j] = src[j];
                    } else {
                        const bf16 *src = L.lw + (size_t)e * r * M + m0 + tid;
                        uint16_t *h = reinterpret_cast<uint16_t *>(ch);
                        for (int q = 0; q < r; ++q) h[q] = *reinterpret_cast<const uint16_t *>(src + (size_t)q * M);
                    }
                }
            }
            for (int sg = 0; sg < pb.nseg; ++sg) {
                const GemmSeg &S = pb.seg[sg];
                const int nkb = S.K / BK;
                const int kmajor = S.kmajor;
                const int kr = tid & 63, half = tid >> 6;
                // K-major: one scale per thread row for the whole tile.  MN-major: one per k-row per k-block (prefetched).
                const __half *scale_p = S.scale + (kmajor ? (size_t)e * M + m0 + tid : (size_t)e * S.K + g * BK + kr);
                __half sc_next = *scale_p;
                uint32_t rowoff, sw;
                if (kmajor) { rowoff = tid * 128; sw = tid & 7; }
                else { rowoff = ((kr >> 3) * 2 + half) * 1024 + (kr & 7) * 128; sw = kr & 7; }
                uint2 codes = make_uint2(0, 0);
                for (int kb = 0; kb < nkb; ++kb) {
                    if ((kb & 1) == 0) {
                        mbar_wait(idx_full(iq.s), iq.ph);
                        const uint32_t is = sbase + OFF_IDX + iq.s * IDX_BYTES;
                        codes = lds64(kmajor ? is + tid * 16 + g * 8 : is + (g * 64 + kr) * 16 + half * 8);
                        __syncwarp();
                        if (lane == 0) mbar_arrive(idx_empty(iq.s));
                        iq.next(IDXQ);
                    }
                    if ((kb & 1) == g) {
                        const __nv_bfloat162 s2 = __float2bfloat162_rn(__half2float(sc_next));
                        if (!kmajor && kb + 2 < nkb) sc_next = scale_p[(kb + 2 - g) * BK];
                        long long tr0 = 0;
                        const bool tr = TQP_DBG(trace != nullptr) && cid == 0 && rank == 0 && threadIdx.x == W_DEQ0 * 32 && dcount < 1000;
                        if (tr) tr0 = clock64();
                        mbar_wait(empty(st.s), st.ph ^ 1);
                        if (tr) { trace[8000 + dcount * 4] = tr0; trace[8000 + dcount * 4 + 1] = clock64(); }
                        const uint32_t as = sbase + OFF_A + st.s * A_BYTES + rowoff;
                        const uint32_t c01[2] = {codes.x, codes.y};
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const uint32_t code = (c01[j >> 2] >> ((j & 3) * 8)) & 0xffu;
                            uint4 v = TQP_DBG(ablate & 1) ? make_uint4(code, code, code, code) : lds128(lut_a + code * 128);
                            __nv_bfloat162 *pv = reinterpret_cast<__nv_bfloat162 *>(&v);
                            if (!TQP_DBG(ablate & 4)) {
#pragma unroll
                                for (int q = 0; q < 4; ++q) pv[q] = __hmul2(pv[q], s2);
                            }
                            if (!TQP_DBG(ablate & 2)) sts128(as + ((j ^ sw) << 4), v);
                        }
                        if (tr) trace[12000 + dcount * 2] = clock64();
                        if (!TQP_DBG(ablate & 128)) fence_async_smem();
                        if (tr) trace[8000 + dcount * 4 + 2] = clock64();
                        __syncwarp();
                        if (tr) trace[12000 + dcount * 2 + 1] = clock64();
                        if (lane == 0) mbar_arrive_cluster(full_remote + 8u * st.s);
                        if (tr) { trace[8000 + dcount * 4 + 3] = clock64(); ++dcount; }
                    }
                    st.next(NSTAGE);
                }
            }
            // adapter K-steps: A tile = lw[m0 + tid][0..r) as a K-major row (chunks beyond r zeroed)
            for (int l = 0; l < pb.nlora; ++l) {
                if ((l & 1) == g) {
                    mbar_wait(empty(st.s), st.ph ^ 1);
                    const uint32_t as = sbase + OFF_A + st.s * A_BYTES + tid * 128;
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        if (j < nch) sts128(as + ((j ^ (tid & 7)) << 4), ch[j]);
                    fence_async_smem();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(full_remote + 8u * st.s);
                }
                st.next(NSTAGE);
            }
        }
    } else if (warp >= W_EPI0) {
        // =========================== epilogue (128 threads) ===========================
        // TMEM (lane = output channel, column = routed row) -> registers in the fragment layout -> bf16 ->
        // stmatrix.trans into a [32 rows][128 channels] staging tile (16-byte chunks XOR-swizzled by row) ->
        // 16-byte coalesced global stores (a half-warp writes one 256-byte row segment).
        const int q = warp & 3;             // TMEM lane quadrant this warp may access
        const int et = threadIdx.x - W_EPI0 * 32;
        int cnt = 0, gcount = 0;
        for (long long item = cid; item < total; item += ncl) {
            Item it;
            get_item(item, it);
            if (it.t.rows <= 0) continue;
            const GemmProblem &pb = args.p[it.prob];
            const int M = pb.M;
            const int ab = cnt & 1;
            const uint32_t aph = (cnt >> 1) & 1;
            ++cnt;
            mbar_wait(tmem_full(ab), aph);
            tc_fence_after();
            bf16 *outp = pb.out + (size_t)it.t.row0 * M + it.m0;
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + ab * TN;
            for (int c0 = 0; c0 < it.t.rows; c0 += EPI_ROWS, ++gcount) {
                uint32_t v[2][16];
                tmem_ld_16x256b_x4(taddr + c0, v[0]);
                tmem_ld_16x256b_x4(taddr + (16u << 16) + c0, v[1]);
                tmem_ld_wait();
                const uint32_t ebuf = sbase + OFF_EPI + (gcount & 1) * EPI_BYTES;
#pragma unroll
                for (int g8 = 0; g8 < 4; ++g8) {   // 8 routed rows per stmatrix.x4: channels 8j..8j+7 of this warp, j = lane/8
                    const int tok = g8 * 8 + (lane & 7);
                    const uint32_t addr = ebuf + tok * (BM * 2) + (((q * 4 + (lane >> 3)) ^ (tok & 7)) << 4);
                    stsm_x4_t(addr, float2_to_bf16x2(__uint_as_float(v[0][4 * g8]), __uint_as_float(v[0][4 * g8 + 1])),
                              float2_to_bf16x2(__uint_as_float(v[0][4 * g8 + 2]), __uint_as_float(v[0][4 * g8 + 3])),
                              float2_to_bf16x2(__uint_as_float(v[1][4 * g8]), __uint_as_float(v[1][4 * g8 + 1])),
                              float2_to_bf16x2(__uint_as_float(v[1][4 * g8 + 2]), __uint_as_float(v[1][4 * g8 + 3])));
                }
                named_bar_sync(1, 128);   // staging tile complete; also orders the reuse of the other buffer
                if (!TQP_DBG(ablate & 16)) {
#pragma unroll
                    for (int i = 0; i < EPI_ROWS * 16 / 128; ++i) {
                        const int r = et / 16 + 8 * i, ch = et % 16;
                        if (c0 + r < it.t.rows) {
                            const uint4 val = lds128(ebuf + r * (BM * 2) + ((ch ^ (r & 7)) << 4));
                            *reinterpret_cast<uint4 *>(outp + (size_t)(c0 + r) * M + ch * 8) = val;
                        }
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(tmem_empty_remote + 8u * ab);
        }
    }

    __syncwarp();
    tc_fence_before();
    __syncthreads();
    cluster_sync();   // the peer may still read this CTA's smem / signal its barriers until both are done
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc<2>(tmem_base, 512);
    }
}

}  // namespace g2

tqp_status launch_gemm_tcgen05_2cta(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st) {
    for (int i = 0; i < nprob; ++i)
        if (probs[i].M % (2 * g2::BM) != 0) return launch_gemm_tcgen05(c, probs, nprob, st);   // odd number of 128-row tiles
    if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&g2::gemm_tcgen05_2cta_kernel), g2::SMEM_BYTES)) return st_attr;
    GemmArgs args;
    for (int i = 0; i < nprob; ++i) args.p[i] = probs[i];
    args.nprob = nprob;
    const int grid = (c->num_sms / 2) * 2;
    const bool tr = c->trace > 0 && ++c->trace_seq == c->trace;
    g2::gemm_tcgen05_2cta_kernel<<<grid, g2::NTHREADS, g2::SMEM_BYTES, st>>>(
        args, c->p<uint4>(c->ws.lut), c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles), c->ablate, tr ? c->p<long long>(c->ws.trace) : nullptr);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
