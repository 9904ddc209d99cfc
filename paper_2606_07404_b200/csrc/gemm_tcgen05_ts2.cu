// Grouped dequant GEMM on CTA pairs with the weight operand in TENSOR MEMORY, 128-wide A stages (sm_100a) -- the default.
//
//   out[p][m] = sum_seg sum_k act_seg[p][k] * W_seg[m][k]  +  sum_l lact_l[p][q] * lw_l[m][q]
//   W[m][k] = bf16( bf16(codebook[code]) * bf16(scale) )                      (look up, rescale by the norm)
//
// Mapping, operands and epilogue are those of gemm_tcgen05_ts.cu (swap-AB: UMMA M = 256 weight output channels over two
// SMs, N = routed rows of one expert; dequantised A tile written to TMEM with tcgen05.st -- row-wise by the channel's own
// thread in the forward GEMMs, through movmatrix in the backward GEMMs; activations by TMA; one 256-column accumulator
// drained into a bf16 staging tile).  What differs is the granularity of the producer hand-shake: one A stage is 128 k
// (one code-index tile, 64 TMEM columns, two 64-wide activation stages), so the fixed cost per hand-shake (index-tile
// wait, slot wait, tcgen05.wait::st, fence, remote arrive: ~400 of the ~1000 clk a backward producer spent per 64 k) is
// paid half as often.  The backward GEMMs were producer-bound at ~600 clk per 64 k against ~455 clk of MMA issue.
// TMEM: accumulator [0, 256) + 3 A slots of 64 columns.  Barriers: fullB/emptyB per activation stage (TMA <-> MMA),
// fullA/emptyA per A slot (dequant warps <-> MMA), index ring, accumulator full/empty.
//
// Warp roles per CTA (480 threads, 1 CTA/SM, persistent over work items, cluster = 2 CTAs):
//   warp 0  TMA producer of the activation / adapter-projection tiles (signals the LEADER's barrier)
//   warp 1  MMA issuer (leader CTA only, one elected lane) + TMEM allocation; in the PEER CTA the same warp is the item
//           scheduler: it draws item ids from a global counter and publishes them to both CTAs through a 4-deep ring
//   warp 2  TMA producer of the code-index tiles
//   warps 3-10  dequant producers, two groups of four that alternate A stages
//   warps 11-14 epilogue (TMEM -> registers -> bf16 -> staging tile -> 16-byte global stores)
#include "common.cuh"
#include "tc_ptx.cuh"

namespace tqp {
namespace gt2 {
using namespace ptx;

constexpr int BM = 128, BK = 64, TN = kTileRows, HN = kTileRows / 2;
constexpr int AK = 128;                                   // K of one A stage (one index tile, one producer hand-shake) = two B stages
constexpr int NASLOT = 3;                                 // A (weight) slots of 64 TMEM columns
constexpr int X_BYTES = HN * 128;
constexpr int EPI_ROWS = 32, EPI_BYTES = TN * BM * 2;      // staging: the whole [256 rows][128 channels] bf16 output tile
// Shared-memory plan.  SC = false: the vector-quantised format of BASELINE.json (one uint8 code per 8 weights, shared 256 x 8
// codebook, fp16 channel scales).  SC = true: the TurboQuant-MSE format of PAPER.md L944-946 (one uint8 code per rotated
// coordinate, a 256-entry scalar Lloyd-Max table, fp32 row norms): an A stage then needs a 128 x 128-byte code tile instead
// of 128 x 16, so the index ring is 3 deep instead of 8 and the activation ring 4 instead of 6.
template <bool SC>
struct Cfg {
    static constexpr int NSTAGE = SC ? 4 : 6;                 // B (activation) ring
    static constexpr int IDXQ = SC ? 3 : 8;                   // index ring
    static constexpr int IDX_TILE = SC ? 128 * 128 : 128 * 16;
    static constexpr int SCL_BYTES = 128 * 4;                 // 128 values ride with the code tile: fp32 norms (SC), bf16-pair scales (VQ backward), fp16 scales (VQ forward: 256 B)
    static constexpr int IDX_BYTES = SC ? IDX_TILE + 1024 : IDX_TILE + SCL_BYTES;   // SC: 128-byte-swizzled TMA tiles need 1024-byte alignment
    static constexpr int LUT_BYTES = 256 * 8 * 16;            // VQ: 8 replicas of the 16-byte entries; SC: 32 lane-private copies of 4-byte entries
    static constexpr int OFF_X = 0, OFF_LUT = OFF_X + NSTAGE * X_BYTES, OFF_IDX = OFF_LUT + LUT_BYTES,
                         OFF_BAR = OFF_IDX + IDXQ * IDX_BYTES, OFF_EPI = OFF_BAR + 512;
    static constexpr int SMEM_BYTES = OFF_EPI + EPI_BYTES + 1024;
};
constexpr int NTHREADS = 480;
constexpr int W_DEQ0 = 3, W_EPI0 = 11;
constexpr int TM_ACC = 0, TM_A = TN;                      // TMEM columns: accumulator [0, 256), A slots [256, 256 + 64 NASLOT)
// Dynamic item schedule: every CTA pair draws its next item from a global counter (tile-list order = expert order) instead of
// a fixed round-robin share, so no pair runs out of work early.  (Measured, cfg 2 / cfg 3 GEMM time per step on one box:
// static 2.585 / 3.195 ms, dynamic 2.558 / 3.174 ms; with the tile list additionally sorted largest-first 2.565 / 3.275 ms
// -- an item's cost hardly depends on its rows, a 16-row item is dequant-bound and costs ~0.7 of a 256-row one, so there
// is nothing for a longest-first order to balance, and it was dropped.)  The five roles of both CTAs are decoupled (the index
// loader runs about an item ahead of the MMAs, the epilogue an item behind), so ids travel through a ring: the scheduler
// thread (peer CTA, warp 1) writes the id into BOTH CTAs' shared memory and arrives on both `sched_full` barriers; every
// consumer warp of both CTAs arrives on the scheduler's `sched_empty` barrier after it has read the id.  Which pair runs
// which item changes no result: items write disjoint outputs.
constexpr int SQ = 4;                                     // ring depth
constexpr int SCHED_CONSUMERS = 15 + 14;                  // warps that follow the ring: leader 0,1,2,3-10,11-14; peer 0,2,3-10,11-14

struct Item {
    Tile t;
    int prob, m0;
};

// 32 consecutive 32-bit TMEM columns of this thread's lane
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t *v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]),
        "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]),
        "r"(v[21]), "r"(v[22]), "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]),
        "r"(v[31])
        : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t *v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]),
        "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}


template <bool SC>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
gemm_tcgen05_ts2_kernel(const __grid_constant__ GemmArgs args, const uint4 *__restrict__ lut_g, const Tile *__restrict__ tiles,
                        const int32_t *__restrict__ num_tiles_p, int32_t *__restrict__ sched_counter, int ablate,
                        long long *__restrict__ trace) {
    using C = Cfg<SC>;
    constexpr int NSTAGE = C::NSTAGE, IDXQ = C::IDXQ, IDX_TILE = C::IDX_TILE, SCL_BYTES = C::SCL_BYTES, IDX_BYTES = C::IDX_BYTES;
    constexpr int OFF_X = C::OFF_X, OFF_LUT = C::OFF_LUT, OFF_IDX = C::OFF_IDX, OFF_BAR = C::OFF_BAR, OFF_EPI = C::OFF_EPI;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar0 = sbase + OFF_BAR;
    auto fullB = [&](int s) { return bar0 + 8u * s; };                               // the LEADER's: expect_tx + 2 x X_BYTES of TMA
    auto emptyB = [&](int s) { return bar0 + 8u * (NSTAGE + s); };                   // local, multicast commit
    auto fullA = [&](int s) { return bar0 + 8u * (2 * NSTAGE + s); };                // the LEADER's: 8 dequant-warp arrivals
    auto emptyA = [&](int s) { return bar0 + 8u * (2 * NSTAGE + NASLOT + s); };      // local, multicast commit
    auto idx_full = [&](int s) { return bar0 + 8u * (2 * NSTAGE + 2 * NASLOT + s); };            // local
    auto idx_empty = [&](int s) { return bar0 + 8u * (2 * NSTAGE + 2 * NASLOT + IDXQ + s); };    // local, the owning group's 4 warps
    const uint32_t tmem_full = bar0 + 8u * (2 * NSTAGE + 2 * NASLOT + 2 * IDXQ);       // local, multicast commit
    const uint32_t tmem_empty = bar0 + 8u * (2 * NSTAGE + 2 * NASLOT + 2 * IDXQ + 1);  // the leader's is used
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + OFF_BAR + 8 * (2 * NSTAGE + 2 * NASLOT + 2 * IDXQ + 4));
    constexpr int NB0 = 2 * NSTAGE + 2 * NASLOT + 2 * IDXQ + 6;
    auto sched_full = [&](int s) { return bar0 + 8u * (NB0 + s); };                  // local: one arrival by the scheduler
    auto sched_empty = [&](int s) { return bar0 + 8u * (NB0 + SQ + s); };            // the PEER's (rank 1) is used
    const uint32_t sched_item = bar0 + 8u * (NB0 + 2 * SQ);                          // SQ ints, a copy in each CTA
    static_assert(8 * (NB0 + 2 * SQ) + 4 * SQ <= 512, "barrier area");

    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const uint32_t rank = cluster_ctarank();
    const uint32_t fullB_remote = mapa(fullB(0), 0), fullA_remote = mapa(fullA(0), 0), tmem_empty_remote = mapa(tmem_empty, 0);
    const uint32_t sched_empty_remote = mapa(sched_empty(0), 1);

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) { mbar_init(fullB(s), 1); mbar_init(emptyB(s), 1); }
        for (int s = 0; s < NASLOT; ++s) { mbar_init(fullA(s), 8); mbar_init(emptyA(s), 1); }
        for (int s = 0; s < IDXQ; ++s) { mbar_init(idx_full(s), 1); mbar_init(idx_empty(s), 4); }
        mbar_init(tmem_full, 1);
        mbar_init(tmem_empty, 8);
        for (int s = 0; s < SQ; ++s) { mbar_init(sched_full(s), 1); mbar_init(sched_empty(s), SCHED_CONSUMERS); }
        mbar_init_fence();
    }
    if (warp == 1) tmem_alloc<2>(smem_u32(tmem_slot), 512);
    if (!SC) {   // replicated LUT: entry e, copy c at (e*8 + c) * 16 B  ->  lane c of every quarter-warp hits bank group c
        uint4 *lut_s = reinterpret_cast<uint4 *>(smem + OFF_LUT);
        for (int i = threadIdx.x; i < 256 * 8; i += NTHREADS) lut_s[i] = lut_g[i >> 3];
    } else {     // scalar table: level e (bf16, low half of a word), one copy per lane at (e * 32 + lane) * 4 B: bank = lane, never a conflict
        uint32_t *lut_s = reinterpret_cast<uint32_t *>(smem + OFF_LUT);
        const uint16_t *lv = reinterpret_cast<const uint16_t *>(lut_g);
        for (int i = threadIdx.x; i < 256 * 32; i += NTHREADS) lut_s[i] = lv[i >> 5];
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync();   // both CTAs' barriers are initialised before any remote arrive / TMA completion
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int num_tiles = *num_tiles_p;
    const int nprob = args.nprob;
    const int MTP = args.p[0].M / (2 * BM);
    const int total = num_tiles * nprob * MTP;
    const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;
    // next item id of this CTA pair (-1: none left); `sq` is the caller's ring position.  _thread: called by ONE thread of
    // a warp (the single-thread roles); _warp: by all 32 lanes.
    auto next_item_thread = [&](Pipe &sq) {
        mbar_wait(sched_full(sq.s), sq.ph);
        const uint32_t v = lds32(sched_item + 4u * sq.s);
        mbar_arrive_cluster_after(sched_empty_remote + 8u * sq.s, v);
        sq.next(SQ);
        return (int)v;
    };
    auto next_item_warp = [&](Pipe &sq) {
        mbar_wait(sched_full(sq.s), sq.ph);
        const uint32_t v = lds32(sched_item + 4u * sq.s);
        const uint32_t all = __reduce_or_sync(0xffffffffu, v);   // every lane's read has returned (all lanes read the same word)
        if (lane == 0) mbar_arrive_cluster_after(sched_empty_remote + 8u * sq.s, all);
        sq.next(SQ);
        return (int)v;
    };

    auto get_item = [&](int item, Item &it) {
        const int tile_id = (int)(item / (nprob * MTP)), rem = (int)(item % (nprob * MTP));
        it.t = tiles[tile_id];
        it.prob = rem / MTP;
        it.m0 = ((rem % MTP) * 2 + (int)rank) * BM;
    };

    if (warp == 0) {
        // =========================== activation TMA producer ===========================
        if (lane == 0) {
            Pipe st, sq;
            for (int item; (item = next_item_thread(sq)) >= 0;) {
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
                        mbar_wait(emptyB(st.s), st.ph ^ 1);
                        if (TQP_DBG(ablate & 64)) {   // timing experiment: no activation traffic (the MMAs read stale tiles)
                            if (rank == 0) mbar_arrive(fullB(st.s));
                            st.next(NSTAGE);
                            continue;
                        }
                        if (rank == 0) mbar_expect_tx(fullB(st.s), 2 * X_BYTES);
                        tma_load_2d_pair(sbase + OFF_X + st.s * X_BYTES, &S.act_map2, kb * BK, row, fullB_remote + 8u * st.s);
                        st.next(NSTAGE);
                    }
                }
                for (int l = 0; l < pb.nlora; ++l) {
                    mbar_wait(emptyB(st.s), st.ph ^ 1);
                    if (rank == 0) mbar_expect_tx(fullB(st.s), 2 * X_BYTES);
                    tma_load_2d_pair(sbase + OFF_X + st.s * X_BYTES, &pb.lora[l].lact_map2, 0, row, fullB_remote + 8u * st.s);
                    st.next(NSTAGE);
                }
            }
        }
    } else if (warp == 2) {
        // =========================== code-index TMA producer ===========================
        if (lane == 0) {
            Pipe iq, sq;
            for (int item; (item = next_item_thread(sq)) >= 0;) {
                Item it;
                get_item(item, it);
                if (it.t.rows <= 0) continue;
                const GemmProblem &pb = args.p[it.prob];
                // This thread runs about one item ahead of the dequant warps: it pulls the item's adapter rows (read once per
                // step, so cold in HBM) into L2 now; fetched cold by the producers they cost an HBM round trip.
                for (int l = 0; l < pb.nlora; ++l) {
                    const GemmLora &L = pb.lora[l];
                    if (L.mk_layout) {
                        const char *p0 = reinterpret_cast<const char *>(L.lw + ((size_t)it.t.expert * pb.M + it.m0) * pb.r);
                        for (int off = 0; off < BM * pb.r * 2; off += 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + off));
                    } else {
                        for (int q = 0; q < pb.r; ++q) {
                            const char *p0 = reinterpret_cast<const char *>(L.lw + ((size_t)it.t.expert * pb.r + q) * pb.M + it.m0);
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(p0));
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + 128));
                        }
                    }
                }
                for (int sg = 0; sg < pb.nseg; ++sg) {
                    const GemmSeg &S = pb.seg[sg];
                    const int nka = S.K / AK;
                    for (int ka = 0; ka < nka; ++ka) {   // K-major: [128 channels][16 codes]; MN-major: [128 k][16 channel groups]
                        mbar_wait(idx_empty(iq.s), iq.ph ^ 1);
                        const uint32_t scl_bytes = (SC || !S.kmajor) ? SCL_BYTES : 256u;
                        mbar_expect_tx(idx_full(iq.s), IDX_TILE + scl_bytes);
                        // VQ: a code covers 8 weights along the pack's input dim; SC: one code per weight
                        const int c0 = S.kmajor ? ka * (SC ? AK : AK / 8) : (SC ? it.m0 : it.m0 / 8);
                        const int c1 = S.kmajor ? it.t.expert * pb.M + it.m0 : it.t.expert * S.K + ka * AK;
                        tma_load_2d(sbase + OFF_IDX + iq.s * IDX_BYTES, &S.idx_map, c0, c1, idx_full(iq.s));
                        // the stage's scales ride along (K-major: of this CTA's 128 channels; MN-major: of the stage's 128 k), so
                        // that no producer waits on a global load when an item starts
                        if (SC) bulk_g2s(sbase + OFF_IDX + iq.s * IDX_BYTES + IDX_TILE, S.norm + c1, SCL_BYTES, idx_full(iq.s));
                        else if (S.kmajor) bulk_g2s(sbase + OFF_IDX + iq.s * IDX_BYTES + IDX_TILE, S.scale + c1, 256u, idx_full(iq.s));
                        else bulk_g2s(sbase + OFF_IDX + iq.s * IDX_BYTES + IDX_TILE, S.scale2 + c1, SCL_BYTES, idx_full(iq.s));   // bf16 pairs, ready to multiply
                        iq.next(IDXQ);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer (leader CTA) ===========================
        if (rank == 1) {
            // =========================== item scheduler (peer CTA) ===========================
            if (elect_one()) {
                Pipe sq;
                const uint32_t item_r0 = mapa(sched_item, 0), full_r0 = mapa(sched_full(0), 0);
                const uint32_t item_r1 = mapa(sched_item, 1), full_r1 = mapa(sched_full(0), 1);
                for (;;) {
                    mbar_wait(sched_empty(sq.s), sq.ph ^ 1);   // every consumer warp of both CTAs has read the entry's previous id
                    const int f = atomicAdd(sched_counter, 1);
                    const int v = f < total ? f : -1;
                    // the id travels as an async store that completes the entry's `full` barrier in each CTA (no fences)
                    mbar_expect_tx_cluster(full_r1 + 8u * sq.s, 4);
                    st_async_u32(item_r1 + 4u * sq.s, (uint32_t)v, full_r1 + 8u * sq.s);
                    mbar_expect_tx_cluster(full_r0 + 8u * sq.s, 4);
                    st_async_u32(item_r0 + 4u * sq.s, (uint32_t)v, full_r0 + 8u * sq.s);
                    if (v < 0) break;
                    sq.next(SQ);
                }
                // the last pair to run dry re-arms the counters for the next launch (stream order: nobody fetches any more)
                if (atomicAdd(sched_counter + 1, 1) == ncl - 1) {
                    sched_counter[0] = 0;
                    sched_counter[1] = 0;
                }
            }
        } else if (elect_one()) {
            Pipe st, sa, sq;
            int cnt = 0;
            const uint32_t hi_k = desc_hi(1024), lo_k = desc_lo_const(16);          // K-major SW128: SBO = 8 rows x 128 B
            const uint32_t x16 = (sbase + OFF_X) >> 4;
            for (int item; (item = next_item_thread(sq)) >= 0;) {
                Item it;
                get_item(item, it);
                if (it.t.rows <= 0) continue;
                const GemmProblem &pb = args.p[it.prob];
                const uint32_t aph = cnt & 1;
                ++cnt;
                const int n = max(16, (it.t.rows + 15) & ~15);
                const bool trc = TQP_DBG(trace != nullptr) && cid == 0 && cnt <= 400;   // per item: start | accumulator free | first operands | per-stage waits | end
                long long ts0 = 0, ts1 = 0, ts2 = 0, twait = 0, twaitb = 0;
                if (trc) ts0 = clock64();
                mbar_wait<true>(tmem_empty, aph ^ 1);   // the epilogue has drained the previous item's accumulator
                tc_fence_after();
                if (trc) ts1 = clock64();
                const uint32_t d_tmem = tmem_base + TM_ACC;
                const uint32_t idesc = make_idesc(2 * BM, n, 0);
                uint32_t accum = 0;
                int nka = 0;
                for (int sg = 0; sg < pb.nseg; ++sg) nka += pb.seg[sg].K / AK;
                const int nmma_l = max(1, pb.r / 16);
                for (int ja = 0; ja < nka + pb.nlora; ++ja) {
                    const bool lora = ja >= nka;
                    long long tw0 = 0;
                    if (trc) tw0 = clock64();
                    mbar_wait<true>(fullA(sa.s), sa.ph);
                    long long twa = 0;
                    if (trc) twa = clock64();
                    const uint32_t a_tmem = tmem_base + TM_A + sa.s * 64;
                    for (int h = 0; h < (lora ? 1 : 2); ++h) {
                        long long twb = 0;
                        if (trc && h == 1) twb = clock64();
                        mbar_wait<true>(fullB(st.s), st.ph);
                        tc_fence_after();
                        if (trc && h == 0) {
                            const long long tw1 = clock64();
                            if (ja == 0) ts2 = tw1; else { twait += twa - tw0; twaitb += tw1 - twa; }
                        }
                        if (trc && h == 1) twaitb += clock64() - twb;
                        const uint32_t xs = x16 + st.s * (X_BYTES >> 4);
                        if (!lora) {
#pragma unroll
                            for (int kk = 0; kk < BK / 16; ++kk) {
                                umma_bf16_ts<2>(d_tmem, a_tmem + h * 32 + kk * 8, desc_from(hi_k, lo_k, xs + kk * 2), idesc, accum);
                                accum = 1;
                            }
                        } else {
                            for (int kk = 0; kk < nmma_l; ++kk) {
                                umma_bf16_ts<2>(d_tmem, a_tmem + kk * 8, desc_from(hi_k, lo_k, xs + kk * 2), idesc, accum);
                                accum = 1;
                            }
                        }
                        umma_commit_pair(emptyB(st.s), 3);
                        st.next(NSTAGE);
                    }
                    umma_commit_pair(emptyA(sa.s), 3);
                    sa.next(NASLOT);
                }
                umma_commit_pair(tmem_full, 3);
                if (trc) {
                    long long *tp = trace + (cnt - 1) * 8;
                    tp[0] = ts0; tp[1] = ts1; tp[2] = ts2; tp[3] = twait; tp[4] = clock64(); tp[5] = nka + pb.nlora; tp[6] = twaitb;
                }
            }
        }
    } else if (warp >= W_DEQ0 && warp < W_EPI0) {
        // =========================== dequant producers: 2 groups x 128 threads ===========================
        // A stage ja (128 k, counted over the whole run of this cluster) belongs to group ja % 2 and to A slot ja % 3.
        const int g = (warp - W_DEQ0) >> 2;
        const int row = (warp & 3) * 32 + lane;                       // K-major: this thread's channel = its TMEM lane
        const uint32_t lut_a = sbase + OFF_LUT + (lane & 7) * 16;
        const uint32_t a_lane = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + TM_A;
        const int rk = lane >> 2, jj = lane & 3;                       // MN-major: source row / channel pair of a movmatrix block
        const int kofs = 4 * (rk >> 1) + (rk & 1);
        const uint32_t lut_b = sbase + OFF_LUT + rk * 16 + jj * 4;   // replica rk: all 32 lanes hit distinct banks
        Pipe sa, iq, sq;
        int ja = 0;
        auto wait_slot_free = [&]() {   // MMAs of the previous use of this A slot have completed
            mbar_wait(emptyA(sa.s), sa.ph ^ 1);
            tc_fence_after();
        };
        auto publish = [&]() {          // the A stage is in TMEM: tell the MMA issuer (the leader CTA's barrier)
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(fullA_remote + 8u * sa.s);
        };
        for (int item; (item = next_item_warp(sq)) >= 0;) {
            Item it;
            get_item(item, it);
            if (it.t.rows <= 0) continue;
            const GemmProblem &pb = args.p[it.prob];
            const int m0 = it.m0, M = pb.M, e = it.t.expert;
            int nka_tot = 0;
            for (int sg = 0; sg < pb.nseg; ++sg) nka_tot += pb.seg[sg].K / AK;
            // adapter row of this channel for the item's last K-step(s): fetched now, consumed after the k-loop
            const int r = pb.r;
            uint32_t ch[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) ch[j] = 0;
            for (int l = 0; l < pb.nlora; ++l) {
                if (((ja + nka_tot + l) & 1) == g) {
                    // all loads of the row are issued back to back (fixed trip counts, predicated on r)
                    const GemmLora &L = pb.lora[l];
                    if (L.mk_layout) {
                        const uint4 *src = reinterpret_cast<const uint4 *>(L.lw + ((size_t)e * M + m0 + row) * r);
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            if (8 * j < r) {
                                const uint4 v = src[j];
                                ch[4 * j] = v.x; ch[4 * j + 1] = v.y; ch[4 * j + 2] = v.z; ch[4 * j + 3] = v.w;
                            }
                        }
                    } else {
                        const uint16_t *src = reinterpret_cast<const uint16_t *>(L.lw + (size_t)e * r * M + m0 + row);
                        uint32_t lo[16], hi[16];
#pragma unroll
                        for (int q = 0; q < 16; ++q) {
                            lo[q] = 2 * q < r ? src[(size_t)(2 * q) * M] : 0u;
                            hi[q] = 2 * q + 1 < r ? src[(size_t)(2 * q + 1) * M] : 0u;
                        }
#pragma unroll
                        for (int q = 0; q < 16; ++q) ch[q] = lo[q] | (hi[q] << 16);
                    }
                    if (pb.seg[0].kmajor) {
                        // Forward items keep the channel scale OUT of the mainloop: the accumulator holds sum_k x[k] bf16(cb)[m][k]
                        // and the epilogue multiplies lane m by the exact fp32 scale (one rounding of the weight instead of
                        // three).  The adapter K-step shares that accumulator, so its row goes in divided by the scale.
                        // (A channel whose scale is 0 -- a zero weight row -- has no base term: its producer writes zeros, the
                        // epilogue multiplies by 1 and the adapter row goes in as it is.)
                        const float scl = SC ? pb.seg[0].norm[(size_t)e * M + m0 + row] : __half2float(pb.seg[0].scale[(size_t)e * M + m0 + row]);
                        const float inv = scl != 0.f ? 1.f / scl : 1.f;
#pragma unroll
                        for (int q = 0; q < 16; ++q) {
                            const float2 f = bf16x2_to_float2(ch[q]);
                            ch[q] = float2_to_bf16x2(f.x * inv, f.y * inv);
                        }
                    }
                }
            }
            for (int sg = 0; sg < pb.nseg; ++sg) {
                const GemmSeg &S = pb.seg[sg];
                const int nka = S.K / AK;
                if (SC && S.kmajor) {
                    // ---- TurboQuant forward: one code per coordinate.  This thread owns channel `row` (its TMEM lane) and
                    // looks its 128 codes of the stage up one by one in its lane-private copy of the scalar table; the tile
                    // row is 128 bytes, its 16-byte chunks XOR-swizzled by row (TMA SWIZZLE_128B), so the LDS.128 of the 32
                    // lanes spread over all banks.  The operand is bf16(level[code]); the row norm multiplies the accumulator lane in the epilogue.
                    const uint32_t lut_l = sbase + OFF_LUT + lane * 4;
                    for (int ka = 0; ka < nka; ++ka) {
                        const bool own = (ja & 1) == g;
                        if (own) {
                            mbar_wait(idx_full(iq.s), iq.ph);
                            const uint32_t tb = sbase + OFF_IDX + iq.s * IDX_BYTES;
                            const bool zero_row = lds32(tb + IDX_TILE + row * 4) << 1 == 0;   // norm 0: no base term for this channel
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                uint32_t a[32];   // 64 bf16 of this channel's row = 32 TMEM columns
#pragma unroll
                                for (int j = 0; j < 4; ++j) {
                                    const uint4 cq = lds128(tb + row * 128 + (((4 * h + j) ^ (row & 7)) << 4));
                                    const uint32_t cw4[4] = {cq.x, cq.y, cq.z, cq.w};
#pragma unroll
                                    for (int w = 0; w < 4; ++w) {
                                        uint32_t lv[4];
#pragma unroll
                                        for (int b = 0; b < 4; ++b) lv[b] = lds32(lut_l + (__byte_perm(cw4[w], 0, 0x4440 | b) << 7));
#pragma unroll
                                        for (int pr = 0; pr < 2; ++pr)   // the row norm is applied by the epilogue (fp32)
                                            a[8 * j + 2 * w + pr] = __byte_perm(lv[2 * pr], lv[2 * pr + 1], 0x5410);
                                    }
                                }
                                if (zero_row) {
#pragma unroll
                                    for (int j = 0; j < 32; ++j) a[j] = 0;
                                }
                                if (h == 1) {   // all codes of the stage are in registers: hand the ring entry back
                                    __syncwarp();
                                    if (lane == 0) mbar_arrive(idx_empty(iq.s));
                                }
                                if (h == 0) wait_slot_free();
                                tmem_st32(a_lane + sa.s * 64 + h * 32, a);
                            }
                            publish();
                        }
                        iq.next(IDXQ);
                        sa.next(NASLOT);
                        ++ja;
                    }
                } else if (SC) {
                    // ---- TurboQuant backward: the contraction runs across the code rows (k = the pack's output channel, whose
                    // norm scales the row); thread (rk, jj) of quadrant q fetches, for each of its 16 k, the code PAIRS of
                    // channels 32 q + 8 cg + 2 jj (+1), cg = 0..3, looks both up and hands the bf16 pair to movmatrix exactly
                    // like the vector-quantised path below.  Tile: 128 k rows of 128 bytes, chunks swizzled by k.
                    const uint32_t lut_l = sbase + OFF_LUT + lane * 4;
                    const int q4 = warp & 3;
                    __nv_bfloat162 sc[16];
                    for (int ka = 0; ka < nka; ++ka) {
                        const bool own = (ja & 1) == g;
                        if (own) {
                            mbar_wait(idx_full(iq.s), iq.ph);
                            const uint32_t tb = sbase + OFF_IDX + iq.s * IDX_BYTES;
#pragma unroll
                            for (int z = 0; z < 16; ++z) {
                                const int kz = (z >> 3) * 64 + ((z >> 1) & 3) * 16 + (z & 1) * 2;
                                sc[z] = __float2bfloat162_rn(__uint_as_float(lds32(tb + IDX_TILE + (kz + kofs) * 4)));
                            }
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
#pragma unroll
                                for (int hs = 0; hs < 2; ++hs) {
                                    uint32_t rg[16];
#pragma unroll
                                    for (int x = 0; x < 4; ++x)
#pragma unroll
                                        for (int mbi = 0; mbi < 2; ++mbi) {
                                            // The eight source rows of a movmatrix block are k0 + {0,1,4,5,8,9,12,13}: rows rk and rk + 4 share
                                            // k & 7, hence the chunk the 128-byte swizzle puts their codes in, hence their banks.  The upper
                                            // half-warp therefore fetches its i = 1 codes while the lower one fetches i = 0 (k & 7 then
                                            // takes all eight values) and the two results are swapped back before the transposition.
                                            const int cg = 2 * hs + mbi;
                                            uint32_t pk[2];
#pragma unroll
                                            for (int pass = 0; pass < 2; ++pass) {
                                                const int k = 64 * h + 16 * x + 2 * (pass ^ (rk >> 2)) + kofs;
                                                // byte column m = 32 q + 8 cg + 2 jj: chunk 2 q + cg / 2, offset 8 (cg % 2) + 2 jj
                                                const uint32_t cp = lds16(tb + k * 128 + (((2 * q4 + (cg >> 1)) ^ (k & 7)) << 4) + 8 * (cg & 1) + 2 * jj);
                                                const uint32_t l0 = lds32(lut_l + ((cp & 0xffu) << 7));
                                                const uint32_t l1 = lds32(lut_l + ((cp >> 8) << 7));
                                                pk[pass] = __byte_perm(l0, l1, 0x5410);
                                            }
#pragma unroll
                                            for (int i = 0; i < 2; ++i) {
                                                const int z = 8 * h + 2 * x + i;
                                                uint32_t p = (rk >> 2) ? pk[i ^ 1] : pk[i];
                                                __nv_bfloat162 w2 = __hmul2(*reinterpret_cast<__nv_bfloat162 *>(&p), sc[z]);
                                                rg[4 * x + 2 * mbi + i] = movmatrix_t(*reinterpret_cast<uint32_t *>(&w2));
                                            }
                                        }
                                    if (h == 1 && hs == 1) {
                                        __syncwarp();
                                        if (lane == 0) mbar_arrive(idx_empty(iq.s));
                                    }
                                    if (h == 0 && hs == 0) wait_slot_free();
                                    tmem_st_16x256b_x4(a_lane + ((uint32_t)(16 * hs) << 16) + sa.s * 64 + h * 32, rg);
                                }
                            }
                            publish();
                        }
                        iq.next(IDXQ);
                        sa.next(NASLOT);
                        ++ja;
                    }
                } else if (S.kmajor) {
                    // ---- forward: codes run along k; this thread owns TMEM lane `row` and writes its 128 k-values itself
                    for (int ka = 0; ka < nka; ++ka) {
                        const bool own = (ja & 1) == g;
                        uint4 codes = make_uint4(0, 0, 0, 0);
                        uint32_t sraw = 0;
                        if (own) {   // one index tile = 16 codes per channel = this A stage
                            mbar_wait(idx_full(iq.s), iq.ph);
                            codes = lds128(sbase + OFF_IDX + iq.s * IDX_BYTES + row * 16);
                            sraw = lds16(sbase + OFF_IDX + iq.s * IDX_BYTES + IDX_TILE + row * 2);
                            __syncwarp();
                            if (lane == 0) mbar_arrive(idx_empty(iq.s));
                        }
                        iq.next(IDXQ);
                        if (own) {
                            // the channel scale is applied by the epilogue (fp32, exact); here it only matters whether it is zero
                            const uint32_t cwd[4] = {codes.x, codes.y, codes.z, codes.w};
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                uint32_t a[32];   // 64 bf16 of this channel's row = 32 TMEM columns
#pragma unroll
                                for (int j = 0; j < 8; ++j) {
                                    const uint32_t code = __byte_perm(cwd[2 * h + (j >> 2)], 0, 0x4440 | (j & 3));   // one PRMT
                                    const uint4 v = lds128(lut_a + code * 128);
                                    a[4 * j] = v.x; a[4 * j + 1] = v.y; a[4 * j + 2] = v.z; a[4 * j + 3] = v.w;
                                }
                                if ((sraw & 0x7fffu) == 0) {   // zero scale: no base term for this channel
#pragma unroll
                                    for (int j = 0; j < 32; ++j) a[j] = 0;
                                }
                                if (h == 0) wait_slot_free();
                                tmem_st32(a_lane + sa.s * 64 + h * 32, a);
                            }
                            publish();
                        }
                        sa.next(NASLOT);
                        ++ja;
                    }
                } else {
                    // ---- backward: codes run along the OUTPUT channels; one codebook row holds 8 channels of one k.
                    // Thread t = (rk = t / 4, jj = t % 4) gathers 4-byte pieces (2 channels) of the rows of its k-values, and
                    // movmatrix turns each 8 (k) x 8 (channel) block into the accumulator-fragment layout of
                    // tcgen05.st.16x256b: lane = channel, register = k pair.  Source row rk of a block carries
                    // k = 16 x + 4 (rk / 2) + rk % 2 + 2 i, so that the transposed pairs land in TMEM columns 8 x + 2 jj + i.
                    uint32_t cw[16];             // code words (4 channel groups each) of this thread's 16 k-values of its A stage
                    __nv_bfloat162 sc[16];       // and their per-k scales (the weight's output channel is k here)
                    for (int ka = 0; ka < nka; ++ka) {
                        const bool own = (ja & 1) == g;
                        if (own) {   // one index tile = 128 k x 16 channel groups = this A stage
                            mbar_wait(idx_full(iq.s), iq.ph);
                            const uint32_t is = sbase + OFF_IDX + iq.s * IDX_BYTES + kofs * 16 + (warp & 3) * 4;
                            const uint32_t ss = sbase + OFF_IDX + iq.s * IDX_BYTES + IDX_TILE + kofs * 4;   // the stage's per-k scales as bf16 pairs
#pragma unroll
                            for (int z = 0; z < 16; ++z) {   // z = 8 h + 2 x + i  ->  k = 64 h + 16 x + kofs + 2 i
                                const int kz = (z >> 3) * 64 + ((z >> 1) & 3) * 16 + (z & 1) * 2;
                                cw[z] = lds32(is + kz * 16);
                                const uint32_t sv = lds32(ss + kz * 4);
                                sc[z] = *reinterpret_cast<const __nv_bfloat162 *>(&sv);
                            }
                            __syncwarp();
                            if (lane == 0) mbar_arrive(idx_empty(iq.s));
                        }
                        iq.next(IDXQ);
                        if (own) {
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
#pragma unroll
                                for (int hs = 0; hs < 2; ++hs) {   // lanes +0..15 / +16..31 of this warp's quadrant
                                    uint32_t rg[16];
#pragma unroll
                                    for (int x = 0; x < 4; ++x)
#pragma unroll
                                        for (int i = 0; i < 2; ++i)
#pragma unroll
                                            for (int mbi = 0; mbi < 2; ++mbi) {
                                                const int z = 8 * h + 2 * x + i;
                                                const uint32_t code = __byte_perm(cw[z], 0, 0x4440 | (2 * hs + mbi));   // one PRMT
                                                uint32_t v = lds32(lut_b + code * 128);
                                                __nv_bfloat162 w2 = __hmul2(*reinterpret_cast<__nv_bfloat162 *>(&v), sc[z]);
                                                rg[4 * x + 2 * mbi + i] = movmatrix_t(*reinterpret_cast<uint32_t *>(&w2));
                                            }
                                    if (h == 0 && hs == 0) wait_slot_free();
                                    tmem_st_16x256b_x4(a_lane + ((uint32_t)(16 * hs) << 16) + sa.s * 64 + h * 32, rg);
                                }
                            }
                            publish();
                        }
                        sa.next(NASLOT);
                        ++ja;
                    }
                }
            }
            for (int l = 0; l < pb.nlora; ++l) {
                if ((ja & 1) == g) {
                    wait_slot_free();
                    tmem_st16(a_lane + sa.s * 64, ch);   // columns beyond r/2 are zero
                    publish();
                }
                sa.next(NASLOT);
                ++ja;
            }
        }
    } else if (warp >= W_EPI0) {
        // =========================== epilogue (128 threads) ===========================
        // Drain: TMEM (lane = output channel, column = routed row) -> registers in the fragment layout -> bf16 ->
        // stmatrix.trans into the [rows][128 channels] staging tile (16-byte chunks XOR-swizzled by row); the
        // accumulator is handed back to the MMA issuer as soon as it has been read.  Then 16-byte coalesced global
        // stores (a half-warp writes one 256-byte row segment) overlap the next item's mainloop.
        const int q = warp & 3;             // TMEM lane quadrant this warp may access
        const int et = threadIdx.x - W_EPI0 * 32;
        const uint32_t ebuf = sbase + OFF_EPI;
        int cnt = 0;
        Pipe sq;
        for (int item; (item = next_item_warp(sq)) >= 0;) {
            Item it;
            get_item(item, it);
            if (it.t.rows <= 0) continue;
            const GemmProblem &pb = args.p[it.prob];
            const int M = pb.M;
            const uint32_t aph = cnt & 1;
            ++cnt;
            const bool tre = TQP_DBG(trace != nullptr) && cid == 0 && rank == 0 && et == 0 && cnt <= 400;
            if (tre) trace[4000 + (cnt - 1) * 4] = clock64();
            // forward items: the exact fp32 channel scale (VQ) / row norm (TurboQuant) of this thread's four TMEM lanes
            float esc[2][2] = {{1.f, 1.f}, {1.f, 1.f}};
            if (pb.seg[0].kmajor) {
                const size_t c0 = (size_t)it.t.expert * M + it.m0 + q * 32 + (lane >> 2);
#pragma unroll
                for (int hh = 0; hh < 2; ++hh)
#pragma unroll
                    for (int u = 0; u < 2; ++u)
                    {
                        const float v = SC ? pb.seg[0].norm[c0 + 16 * hh + 8 * u] : __half2float(pb.seg[0].scale[c0 + 16 * hh + 8 * u]);
                        esc[hh][u] = v != 0.f ? v : 1.f;
                    }
            }
            mbar_wait(tmem_full, aph);
            tc_fence_after();
            named_bar_sync(1, 128);   // every epilogue warp has finished storing the previous item out of the staging tile
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + TM_ACC;
            for (int c0 = 0; c0 < it.t.rows; c0 += EPI_ROWS) {
                uint32_t v[2][16];
                tmem_ld_16x256b_x4(taddr + c0, v[0]);
                tmem_ld_16x256b_x4(taddr + (16u << 16) + c0, v[1]);
                tmem_ld_wait();
#pragma unroll
                for (int g8 = 0; g8 < 4; ++g8) {   // 8 routed rows per stmatrix.x4: channels 8j..8j+7 of this warp, j = lane/8
                    const int tok = c0 + g8 * 8 + (lane & 7);
                    const uint32_t addr = ebuf + tok * (BM * 2) + (((q * 4 + (lane >> 3)) ^ (tok & 7)) << 4);
                    stsm_x4_t(addr, float2_to_bf16x2(__uint_as_float(v[0][4 * g8]) * esc[0][0], __uint_as_float(v[0][4 * g8 + 1]) * esc[0][0]),
                              float2_to_bf16x2(__uint_as_float(v[0][4 * g8 + 2]) * esc[0][1], __uint_as_float(v[0][4 * g8 + 3]) * esc[0][1]),
                              float2_to_bf16x2(__uint_as_float(v[1][4 * g8]) * esc[1][0], __uint_as_float(v[1][4 * g8 + 1]) * esc[1][0]),
                              float2_to_bf16x2(__uint_as_float(v[1][4 * g8 + 2]) * esc[1][1], __uint_as_float(v[1][4 * g8 + 3]) * esc[1][1]));
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(tmem_empty_remote);
            if (tre) trace[4000 + (cnt - 1) * 4 + 1] = clock64();
            named_bar_sync(1, 128);   // staging tile complete
            if (!TQP_DBG(ablate & 16)) {
                bf16 *outp = pb.out + (size_t)it.t.row0 * M + it.m0;
                for (int r = et / 16; r < it.t.rows; r += 8) {
                    const int chk = et % 16;
                    const uint4 val = lds128(ebuf + r * (BM * 2) + ((chk ^ (r & 7)) << 4));
                    *reinterpret_cast<uint4 *>(outp + (size_t)r * M + chk * 8) = val;
                }
            }
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

}  // namespace gt2

tqp_status launch_gemm_tcgen05_ts2(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st) {
    const bool sc = probs[0].seg[0].scalar != 0;   // TurboQuant codes (one launch never mixes the two formats)
    for (int i = 0; i < nprob; ++i) {   // an even number of 128-channel tiles and whole 128-wide A stages per segment
        const GemmProblem &p = probs[i];
        bool ok = p.M % (2 * gt2::BM) == 0 && p.nlora <= 2;
        for (int sg = 0; sg < p.nseg; ++sg) ok = ok && p.seg[sg].K % gt2::AK == 0 && (p.seg[sg].scalar != 0) == sc;
        if (!ok) {
            if (sc) { c->err = "TurboQuant-format GEMM needs M % 256 == 0 and K % 128 == 0"; return TQP_ERR_SHAPE; }
            return launch_gemm_tcgen05_2cta(c, probs, nprob, st);
        }
    }
    GemmArgs args;
    for (int i = 0; i < nprob; ++i) args.p[i] = probs[i];
    args.nprob = nprob;
    const int grid = (c->num_sms / 2) * 2;
    const bool tr = c->trace > 0 && ++c->trace_seq == c->trace;   // debug timeline of cluster 0 (-DTQP_TRACE builds)
    int32_t *counter = c->p<int32_t>(c->ws.sched) + 4;
    long long *trace = tr ? c->p<long long>(c->ws.trace) : nullptr;
    if (sc) {
        if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&gt2::gemm_tcgen05_ts2_kernel<true>), gt2::Cfg<true>::SMEM_BYTES)) return st_attr;
        gt2::gemm_tcgen05_ts2_kernel<true><<<grid, gt2::NTHREADS, gt2::Cfg<true>::SMEM_BYTES, st>>>(
            args, reinterpret_cast<const uint4 *>(probs[0].seg[0].lut), c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles), counter, c->ablate, trace);
    } else {
        if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&gt2::gemm_tcgen05_ts2_kernel<false>), gt2::Cfg<false>::SMEM_BYTES)) return st_attr;
        gt2::gemm_tcgen05_ts2_kernel<false><<<grid, gt2::NTHREADS, gt2::Cfg<false>::SMEM_BYTES, st>>>(
            args, c->p<uint4>(c->ws.lut), c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles), counter, c->ablate, trace);
    }
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

}  // namespace tqp
