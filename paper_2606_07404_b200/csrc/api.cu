// C-ABI entry points (include/tqp.h): argument validation, workspace layout, TMA descriptors, call chains.
#include <algorithm>
#include <cstring>
#include <new>

#include "common.cuh"

using namespace tqp;

namespace {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool desc_ok(const tqp_layer_desc *d) {
    if (!d) return false;
    if (d->T_max <= 0 || d->d <= 0 || d->F <= 0 || d->E <= 0 || d->k <= 0) return false;
    if (d->d % 128 || d->F % 128) return false;
    if (d->k > d->E || d->k > 32 || d->E > 1024) return false;
    if (!(d->r == 8 || d->r == 16 || d->r == 32)) return false;
    if (d->vec != 8 || d->codes != 256) return false;
    if ((long long)d->T_max * d->k >= (1ll << 31) / 64) return false;
    return true;
}

Workspace layout(const tqp_layer_desc &d) {
    Workspace w;
    const size_t T = d.T_max, N = T * d.k, Np = N + kRowPad, dm = d.d, F = d.F, E = d.E;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 1024); return o; };
    w.Xp = take(Np * dm * 2);
    w.G = take(Np * F * 2); w.U = take(Np * F * 2); w.H = take(Np * F * 2);
    w.dH = take(Np * F * 2); w.dG = take(Np * F * 2); w.dU = take(Np * F * 2);
    w.XAg = take(Np * kLoraPad * 2); w.XAu = take(Np * kLoraPad * 2); w.HAd = take(Np * kLoraPad * 2);
    w.Zd = take(Np * kLoraPad * 2); w.Zg = take(Np * kLoraPad * 2); w.Zu = take(Np * kLoraPad * 2);
    w.logits = take(T * E * 4);
    w.blk_counts = take(((N + kDispChunk - 1) / kDispChunk + 4) * E * 4);
    w.tiles = take((E + N / kTileRows + 2) * sizeof(Tile));
    w.num_tiles = take(16);
    w.xsegs = take((N / kWgradSeg + 2) * sizeof(Tile));
    w.xfirst = take((E + 1) * 4);
    w.tfirst = take((E + 1) * 4);
    w.sched = take(64);   // work counters of the persistent kernels (zeroed before each launch)
    // partial weight gradients of split experts: first segments indexed by expert, extra segments by list position;
    // widest use: two rank-r gradients over d columns in one pass (dA_gate + dA_up)
    // ... and the per-tile partials of rows_proj_wgrad_kernel: [2][max_tiles][r][F]
    w.wg_scratch = d.training ? take(std::max((E + N / kWgradSeg + 2) * (size_t)2 * d.r * (dm > F ? dm : F) * 4,
                                              (size_t)2 * (E + N / kTileRows + 1) * d.r * F * 4)) : take(16);
    w.wg_done = take(E * ((dm > F ? dm : F) / 128) * 4);   // arrival counters of split experts (rows_wgrad_kernel), zero between launches
    w.lut = take(256 * 8 * 2);
    w.sc2 = take(E * (dm + 2 * F) * 4);   // bf16-pair copies of scale_down | scale_gate | scale_up for the backward GEMMs
    w.WrT = take(E * dm * 4);
    w.WrHL = take(E * dm * 4);   // bf16 hi | lo split of W_r^T, [E][2d] (screened router)
    w.wnorm = take(E * 4);
    w.rflag = take(16);
    w.dl = take(N * 4);
    w.trace = take(16384 * 8);
    w.total = off;
    // Staging of tqp_step_host (X / dY twice, Y, dX, the routing arrays, Ye / dYe / dXp): NOT part of the caller's workspace;
    // the library allocates it on the first tqp_step_host call (a stepwise caller never pays for it: 1.7 GB at cfg 2).
    off = 0;
    w.hX = take(T * dm * 2); w.hdY = take(T * dm * 2); w.hY = take(T * dm * 2); w.hdX = take(T * dm * 2);
    w.hX2 = take(T * dm * 2); w.hdY2 = take(T * dm * 2);   // second upload set (tqp_step_host_async)
    w.topk_idx = take(N * 4); w.topk_w = take(N * 4); w.counts = take(E * 4); w.offsets = take((E + 1) * 4);
    w.perm = take(N * 4); w.inv_perm = take(N * 4);
    w.Ye = take(N * dm * 2); w.dYe = take(N * dm * 2); w.dXp = take(N * dm * 2); w.dtopk_w = take(N * 4);
    w.host_total = off;
    return w;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// 2-D row-major tensor [rows][cols] of `esize`-byte elements, box {box_cols, box_rows}
tqp_status make_map(tqp_ctx *c, CUtensorMap *m, const void *ptr, CUtensorMapDataType dt, size_t esize, uint64_t rows,
                    uint64_t cols, uint32_t box_cols, uint32_t box_rows, CUtensorMapSwizzle sw) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) { c->err = "cuTensorMapEncodeTiled not available"; return TQP_ERR_CUDA; }
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {cols * esize};
    cuuint32_t box[2] = {box_cols, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(m, dt, 2, const_cast<void *>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { c->err = "cuTensorMapEncodeTiled failed: " + std::to_string((int)r); return TQP_ERR_CUDA; }
    return TQP_OK;
}

tqp_status act_map(tqp_ctx *c, CUtensorMap *m, const void *ptr, uint64_t rows, uint64_t K, int box_rows = kTileRows) {
    return make_map(c, m, ptr, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, rows, K, 64, box_rows, CU_TENSOR_MAP_SWIZZLE_128B);
}

// Unswizzled maps of the gathered projections (lora.cu): m[0] = source rows, box {256, 1} (gather4);  m[1], m[2] = the
// permuted destination, box {256, 128} (tile store) and {256, 1} (scatter4 of a ragged tile).
tqp_status gather_maps(tqp_ctx *c, CUtensorMap *m, const void *in, uint64_t in_rows, const void *through, uint64_t out_rows, uint64_t K) {
    const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
    tqp_status st = make_map(c, &m[0], in, dt, 2, in_rows, K, 256, 1, CU_TENSOR_MAP_SWIZZLE_NONE);
    if (st == TQP_OK) st = make_map(c, &m[1], through, dt, 2, out_rows, K, 256, 128, CU_TENSOR_MAP_SWIZZLE_NONE);
    if (st == TQP_OK) st = make_map(c, &m[2], through, dt, 2, out_rows, K, 256, 1, CU_TENSOR_MAP_SWIZZLE_NONE);
    return st;
}

tqp_status set_seg(tqp_ctx *c, GemmSeg *s, const bf16 *act, uint64_t act_rows, const uint8_t *idx, const void *scale, int K,
                   int M, int kmajor) {
    s->act = act; s->idx = idx; s->scale = (const __half *)scale; s->K = K; s->kmajor = kmajor;
    tqp_status st = act_map(c, &s->act_map, act, act_rows, K);
    if (st != TQP_OK) return st;
    st = act_map(c, &s->act_map2, act, act_rows, K, kTileRows / 2);
    if (st != TQP_OK) return st;
    const uint64_t E = c->desc.E;
    const uint64_t rows = kmajor ? E * M : E * K, bytes = kmajor ? K / 8 : M / 8;
    return make_map(c, &s->idx_map, idx, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, rows, bytes, 16, 128, CU_TENSOR_MAP_SWIZZLE_NONE);
}

tqp_status set_lora(tqp_ctx *c, GemmLora *l, const bf16 *lact, uint64_t rows, const void *lw, int mk_layout) {
    l->lact = lact; l->lw = (const bf16 *)lw; l->mk_layout = mk_layout;
    tqp_status st = act_map(c, &l->lact_map2, lact, rows, kLoraPad, kTileRows / 2);
    if (st != TQP_OK) return st;
    return act_map(c, &l->lact_map, lact, rows, kLoraPad);
}

void tq_free_state(tqp_ctx *c);   // defined with the TurboQuant binding below

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

#define REQ(ctx, cond, code, msg)              \
    do {                                       \
        if (!(cond)) {                         \
            (ctx)->err = msg;                  \
            return code;                       \
        }                                      \
    } while (0)

#define PTR_OK(ctx, p)                                                     \
    do {                                                                   \
        REQ(ctx, (p) != nullptr, TQP_ERR_ARG, #p " is NULL");              \
        REQ(ctx, aligned16(p), TQP_ERR_ALIGN, #p " is not 16-byte aligned"); \
    } while (0)

tqp_status common_checks(tqp_ctx *c, int T, bool need_weights) {
    if (!c) return TQP_ERR_ARG;
    c->launches = 0;
    REQ(c, T > 0 && T <= c->desc.T_max, TQP_ERR_ARG, "T out of range (0 < T <= T_max)");
    REQ(c, c->base != nullptr, TQP_ERR_WORKSPACE, "no workspace bound");
    if (need_weights) REQ(c, c->have_weights, TQP_ERR_STATE, "tqp_bind_weights has not been called");
    return TQP_OK;
}

tqp_status run_gemm(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st) {
    const bool timed = c->time_gemm && c->ev_used + 2 <= (int)c->ev.size();
    if (timed) TQP_CUDA_OK(c, cudaEventRecord(c->ev[c->ev_used], st));
    tqp_status r = c->gemm_impl == 1   ? launch_gemm_scaffold(c, probs, nprob, st)
                   : c->gemm_impl == 2 ? launch_gemm_tcgen05(c, probs, nprob, st)
                   : c->gemm_impl == 3 ? launch_gemm_tcgen05_2cta(c, probs, nprob, st)
                                       : launch_gemm_tcgen05_ts2(c, probs, nprob, st);
    if (timed) {
        TQP_CUDA_OK(c, cudaEventRecord(c->ev[c->ev_used + 1], st));
        c->ev_used += 2;
    }
    return r;
}

}  // namespace

extern "C" {

tqp_status tqp_create(tqp_ctx **out, const tqp_layer_desc *desc) {
    if (!out) return TQP_ERR_ARG;
    *out = nullptr;
    if (!desc) return TQP_ERR_ARG;
    if (!desc_ok(desc)) return TQP_ERR_SHAPE;
    int dev = 0, major = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return TQP_ERR_CUDA;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return TQP_ERR_CUDA;
    if (major != 10) return TQP_ERR_ARCH;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    tqp_ctx *c = new (std::nothrow) tqp_ctx();
    if (!c) return TQP_ERR_ARG;
    c->desc = *desc;
    c->device = dev;
    c->ws = layout(*desc);
    c->num_sms = sms > 0 ? sms : 148;
    c->max_tiles = desc->E + (desc->T_max * desc->k) / kTileRows + 1;
    c->max_xsegs = (desc->T_max * desc->k) / kWgradSeg + 1;
    memset(&c->w, 0, sizeof(c->w));
    *out = c;
    return TQP_OK;
}

void tqp_destroy(tqp_ctx *ctx) {
    if (!ctx) return;
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : {ctx->ev_start, ctx->ev_x, ctx->ev_dy, ctx->ev_y, ctx->ev_yout, ctx->ev_dx, ctx->ev_xc[0], ctx->ev_xc[1],
                          ctx->ev_xc[2], ctx->ev_xc[3], ctx->ev_done[0], ctx->ev_done[1], ctx->ev_comp[0], ctx->ev_comp[1]})
        if (e) cudaEventDestroy(e);
    for (auto &r : ctx->tq_rots) { cudaFree(r.Rb); cudaFree(r.Rtb); cudaFree(r.Rt); }
    tq_free_state(ctx);
    if (ctx->host_base) cudaFree(ctx->host_base);
    if (ctx->copy_in) cudaStreamDestroy(ctx->copy_in);
    if (ctx->copy_out) cudaStreamDestroy(ctx->copy_out);
    delete ctx;
}

tqp_status tqp_gemm_times(tqp_ctx *c, float *ms_each, int cap, int *launches) {
    if (!c || !ms_each || !launches) return TQP_ERR_ARG;
    int n = 0;
    for (int i = 0; i + 1 < c->ev_used; i += 2, ++n) {
        TQP_CUDA_OK(c, cudaEventSynchronize(c->ev[i + 1]));
        float ms = 0.f;
        TQP_CUDA_OK(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
        if (n < cap) ms_each[n] = ms;
    }
    *launches = n;
    c->ev_used = 0;
    return TQP_OK;
}

tqp_status tqp_gemm_time(tqp_ctx *c, float *ms_total, int *launches) {
    if (!c || !ms_total || !launches) return TQP_ERR_ARG;
    float total = 0.f;
    for (int i = 0; i + 1 < c->ev_used; i += 2) {
        TQP_CUDA_OK(c, cudaEventSynchronize(c->ev[i + 1]));
        float ms = 0.f;
        TQP_CUDA_OK(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
        total += ms;
    }
    *ms_total = total;
    *launches = c->ev_used / 2;
    c->ev_used = 0;
    return TQP_OK;
}

size_t tqp_workspace_bytes(const tqp_layer_desc *desc) {
    if (!desc_ok(desc)) return 0;
    return layout(*desc).total;
}

tqp_status tqp_bind_workspace(tqp_ctx *c, void *dev_ptr, size_t bytes, void *stream) {
    if (!c) return TQP_ERR_ARG;
    PTR_OK(c, dev_ptr);
    REQ(c, bytes >= c->ws.total, TQP_ERR_WORKSPACE, "workspace too small");
    TQP_CUDA_OK(c, cudaMemsetAsync(dev_ptr, 0, c->ws.total, (cudaStream_t)stream));
    c->base = static_cast<char *>(dev_ptr);
    c->bound_bytes = bytes;
    c->have_weights = false;
    return TQP_OK;
}

tqp_status tqp_bind_weights(tqp_ctx *c, const tqp_weights *w, void *stream) {
    if (!c || !w) return TQP_ERR_ARG;
    REQ(c, c->base != nullptr, TQP_ERR_WORKSPACE, "bind a workspace first");
    const void *ptrs[] = {w->idx_gate, w->idx_up, w->idx_down, w->scale_gate, w->scale_up, w->scale_down, w->codebook,
                          w->A_gate, w->A_up, w->B_gate, w->B_up, w->A_down, w->B_down};
    for (const void *p : ptrs) PTR_OK(c, p);
    c->w = *w;
    c->launches = 0;
    if (c->tq.on) tq_free_state(c);
    const tqp_layer_desc &D = c->desc;
    const uint64_t Np = (uint64_t)D.T_max * D.k + kRowPad;
    tqp_status st = launch_make_lut(c, (const __half *)w->codebook, c->p<bf16>(c->ws.lut), (cudaStream_t)stream);
    if (st != TQP_OK) return st;
    bf16 *Xp = c->p<bf16>(c->ws.Xp), *G = c->p<bf16>(c->ws.G), *U = c->p<bf16>(c->ws.U), *H = c->p<bf16>(c->ws.H);
    bf16 *dH = c->p<bf16>(c->ws.dH), *dG = c->p<bf16>(c->ws.dG), *dU = c->p<bf16>(c->ws.dU);
    GemmProblem *P;
#define CK(x) do { st = (x); if (st != TQP_OK) return st; } while (0)
    P = &c->prob_gate; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.F; P->r = D.r; P->out = G;
    CK(set_seg(c, &P->seg[0], Xp, Np, w->idx_gate, w->scale_gate, D.d, D.F, 1));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.XAg), Np, w->B_gate, 0));
    P = &c->prob_up; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.F; P->r = D.r; P->out = U;
    CK(set_seg(c, &P->seg[0], Xp, Np, w->idx_up, w->scale_up, D.d, D.F, 1));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.XAu), Np, w->B_up, 0));
    P = &c->prob_down; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.d; P->r = D.r; P->out = nullptr;   // out = Ye, per call
    CK(set_seg(c, &P->seg[0], H, Np, w->idx_down, w->scale_down, D.F, D.d, 1));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.HAd), Np, w->B_down, 0));
    uint32_t *sc2_down = c->p<uint32_t>(c->ws.sc2), *sc2_gate = sc2_down + (size_t)D.E * D.d, *sc2_up = sc2_gate + (size_t)D.E * D.F;
    CK(launch_scale_pairs(c, (const __half *)w->scale_down, sc2_down, (size_t)D.E * D.d, (cudaStream_t)stream));
    CK(launch_scale_pairs(c, (const __half *)w->scale_gate, sc2_gate, (size_t)D.E * D.F, (cudaStream_t)stream));
    CK(launch_scale_pairs(c, (const __half *)w->scale_up, sc2_up, (size_t)D.E * D.F, (cudaStream_t)stream));
    P = &c->prob_dh; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.F; P->r = D.r; P->out = dH;       // seg[0].act = dYe, per call
    CK(set_seg(c, &P->seg[0], dH /*placeholder*/, Np, w->idx_down, w->scale_down, D.d, D.F, 0));
    P->seg[0].scale2 = sc2_down;
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.Zd), Np, w->A_down, 1));
    P = &c->prob_dx; memset(P, 0, sizeof(*P));
    P->nseg = 2; P->nlora = 2; P->M = D.d; P->r = D.r; P->out = nullptr;   // out = dXp, per call
    CK(set_seg(c, &P->seg[0], dG, Np, w->idx_gate, w->scale_gate, D.F, D.d, 0));
    CK(set_seg(c, &P->seg[1], dU, Np, w->idx_up, w->scale_up, D.F, D.d, 0));
    P->seg[0].scale2 = sc2_gate; P->seg[1].scale2 = sc2_up;
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.Zg), Np, w->A_gate, 1));
    CK(set_lora(c, &P->lora[1], c->p<bf16>(c->ws.Zu), Np, w->A_up, 1));
#undef CK
    c->have_weights = true;
    return TQP_OK;
}

}  // extern "C"

namespace {

void tq_free_state(tqp_ctx *c) {
    tqp::TqLayer &t = c->tq;
    for (void *p : {(void *)t.Xr, (void *)t.Ar_gate, (void *)t.Ar_up, (void *)t.Ar_down, (void *)t.tmp_a, (void *)t.tmp_b, (void *)t.dAr_gate,
                    (void *)t.dAr_up, (void *)t.dAr_down, (void *)t.tmp_f, (void *)t.lut_d, (void *)t.lut_F})
        if (p) cudaFree(p);
    t = tqp::TqLayer();
}

// scalar-format segment: codes [E][M][K] (kmajor) or used transposed [E][K][M]; box 128 bytes x 128 rows, 128-byte swizzle
tqp_status set_seg_tq(tqp_ctx *c, GemmSeg *s, const bf16 *act, uint64_t act_rows, const uint8_t *codes, const float *norm, const bf16 *lut,
                      int K, int M, int kmajor) {
    s->act = act; s->idx = codes; s->scale = nullptr; s->norm = norm; s->lut = lut; s->scalar = 1; s->K = K; s->kmajor = kmajor;
    tqp_status st = act_map(c, &s->act_map, act, act_rows, K);
    if (st != TQP_OK) return st;
    st = act_map(c, &s->act_map2, act, act_rows, K, kTileRows / 2);
    if (st != TQP_OK) return st;
    const uint64_t E = c->desc.E;
    const uint64_t rows = kmajor ? E * M : E * K, bytes = kmajor ? K : M;
    return make_map(c, &s->idx_map, codes, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, rows, bytes, 128, 128, CU_TENSOR_MAP_SWIZZLE_128B);
}

// A' = R A per expert:  A [E][n][r] -> transpose -> rows [E r][n] -> rotate -> transpose back
tqp_status tq_rotate_adapter(tqp_ctx *c, const tqp_tq_space *sp, const bf16 *A, bf16 *Ar, cudaStream_t s) {
    const int E = c->desc.E, r = c->desc.r, n = sp->n;
    if (sp->hadamard && n <= 8192) return launch_tq_fwht_strided<bf16>(c, sp, A, Ar, E, r, 0, s);   // one pass, no transposes
    tqp_status st = launch_tq_transpose<bf16>(c, A, c->tq.tmp_a, E, n, r, s);
    if (st == TQP_OK) st = launch_tq_rotate(c, sp, c->tq.tmp_a, false, (long long)E * r, c->tq.tmp_b, false, 0, s);
    if (st == TQP_OK) st = launch_tq_transpose<bf16>(c, c->tq.tmp_b, Ar, E, r, n, s);
    return st;
}
// dA = R^T dA' per expert (fp32): the same way back
tqp_status tq_unrotate_grad(tqp_ctx *c, const tqp_tq_space *sp, float *dAr, float *dA, cudaStream_t s) {
    const int E = c->desc.E, r = c->desc.r, n = sp->n;
    if (sp->hadamard && n <= 8192) return launch_tq_fwht_strided<float>(c, sp, dAr, dA, E, r, 1, s);
    tqp_status st = launch_tq_transpose<float>(c, dAr, c->tq.tmp_f, E, n, r, s);
    if (st == TQP_OK) st = launch_tq_rotate(c, sp, c->tq.tmp_f, true, (long long)E * r, dAr, true, 1, s);
    if (st == TQP_OK) st = launch_tq_transpose<float>(c, dAr, dA, E, r, n, s);
    return st;
}

}  // namespace

extern "C" tqp_status tqp_bind_weights_tq(tqp_ctx *c, const tqp_tq_weights *w, void *stream) {
    if (!c || !w) return TQP_ERR_ARG;
    REQ(c, c->base != nullptr, TQP_ERR_WORKSPACE, "bind a workspace first");
    const void *ptrs[] = {w->codes_gate, w->codes_up, w->codes_down, w->norm_gate, w->norm_up, w->norm_down,
                          w->A_gate, w->A_up, w->B_gate, w->B_up, w->A_down, w->B_down};
    for (const void *p : ptrs) PTR_OK(c, p);
    const tqp_layer_desc &D = c->desc;
    tqp_status st = tq_check_space(c, &w->space_d);
    if (st == TQP_OK) st = tq_check_space(c, &w->space_F);
    if (st != TQP_OK) return st;
    REQ(c, w->space_d.n == D.d && w->space_F.n == D.F, TQP_ERR_SHAPE, "space_d.n must be d and space_F.n must be F");
    REQ(c, (D.r == 16 || D.r == 32) && D.d % 256 == 0 && D.F % 256 == 0, TQP_ERR_SHAPE,
        "the TurboQuant-format layer needs r in {16, 32}, d % 256 == 0, F % 256 == 0");
    cudaStream_t s = (cudaStream_t)stream;
    c->launches = 0;
    c->have_weights = false;
    tq_free_state(c);
    tqp::TqLayer &t = c->tq;
    t.w = *w;
    const size_t E = D.E, r = D.r, dm = D.d, F = D.F, mx = dm > F ? dm : F;
    TQP_CUDA_OK(c, cudaMalloc(&t.Xr, (size_t)D.T_max * dm * 2));
    TQP_CUDA_OK(c, cudaMalloc(&t.Ar_gate, E * dm * r * 2)); TQP_CUDA_OK(c, cudaMalloc(&t.Ar_up, E * dm * r * 2));
    TQP_CUDA_OK(c, cudaMalloc(&t.Ar_down, E * F * r * 2));
    TQP_CUDA_OK(c, cudaMalloc(&t.tmp_a, E * mx * r * 2)); TQP_CUDA_OK(c, cudaMalloc(&t.tmp_b, E * mx * r * 2));
    if (D.training) {
        TQP_CUDA_OK(c, cudaMalloc(&t.dAr_gate, E * dm * r * 4)); TQP_CUDA_OK(c, cudaMalloc(&t.dAr_up, E * dm * r * 4));
        TQP_CUDA_OK(c, cudaMalloc(&t.dAr_down, E * F * r * 4)); TQP_CUDA_OK(c, cudaMalloc(&t.tmp_f, E * mx * r * 4));
    }
    TQP_CUDA_OK(c, cudaMalloc(&t.lut_d, 512)); TQP_CUDA_OK(c, cudaMalloc(&t.lut_F, 512));
    st = launch_tq_make_lut(c, w->space_d.levels, t.lut_d, s);
    if (st == TQP_OK) st = launch_tq_make_lut(c, w->space_F.levels, t.lut_F, s);
    if (st != TQP_OK) return st;
    // the adapter pointers of the common code path: B sides as given, A sides replaced by their rotated copies
    memset(&c->w, 0, sizeof(c->w));
    c->w.A_gate = t.Ar_gate; c->w.A_up = t.Ar_up; c->w.A_down = t.Ar_down;
    c->w.B_gate = w->B_gate; c->w.B_up = w->B_up; c->w.B_down = w->B_down;
    const uint64_t Np = (uint64_t)D.T_max * D.k + kRowPad;
    bf16 *Xp = c->p<bf16>(c->ws.Xp), *G = c->p<bf16>(c->ws.G), *U = c->p<bf16>(c->ws.U), *H = c->p<bf16>(c->ws.H);
    bf16 *dH = c->p<bf16>(c->ws.dH), *dG = c->p<bf16>(c->ws.dG), *dU = c->p<bf16>(c->ws.dU);
    GemmProblem *P;
#define CK(x) do { st = (x); if (st != TQP_OK) return st; } while (0)
    P = &c->prob_gate; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.F; P->r = D.r; P->out = G;
    CK(set_seg_tq(c, &P->seg[0], Xp, Np, w->codes_gate, w->norm_gate, t.lut_d, D.d, D.F, 1));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.XAg), Np, w->B_gate, 0));
    P = &c->prob_up; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.F; P->r = D.r; P->out = U;
    CK(set_seg_tq(c, &P->seg[0], Xp, Np, w->codes_up, w->norm_up, t.lut_d, D.d, D.F, 1));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.XAu), Np, w->B_up, 0));
    P = &c->prob_down; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.d; P->r = D.r; P->out = nullptr;
    CK(set_seg_tq(c, &P->seg[0], H, Np, w->codes_down, w->norm_down, t.lut_F, D.F, D.d, 1));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.HAd), Np, w->B_down, 0));
    P = &c->prob_dh; memset(P, 0, sizeof(*P));
    P->nseg = 1; P->nlora = 1; P->M = D.F; P->r = D.r; P->out = dH;
    CK(set_seg_tq(c, &P->seg[0], dH /*placeholder*/, Np, w->codes_down, w->norm_down, t.lut_F, D.d, D.F, 0));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.Zd), Np, t.Ar_down, 1));
    P = &c->prob_dx; memset(P, 0, sizeof(*P));
    P->nseg = 2; P->nlora = 2; P->M = D.d; P->r = D.r; P->out = nullptr;
    CK(set_seg_tq(c, &P->seg[0], dG, Np, w->codes_gate, w->norm_gate, t.lut_d, D.F, D.d, 0));
    CK(set_seg_tq(c, &P->seg[1], dU, Np, w->codes_up, w->norm_up, t.lut_d, D.F, D.d, 0));
    CK(set_lora(c, &P->lora[0], c->p<bf16>(c->ws.Zg), Np, t.Ar_gate, 1));
    CK(set_lora(c, &P->lora[1], c->p<bf16>(c->ws.Zu), Np, t.Ar_up, 1));
#undef CK
    t.on = true;
    c->have_weights = true;
    return TQP_OK;
}

extern "C" {

tqp_status tqp_set_option(tqp_ctx *c, const char *name, int value) {
    if (!c || !name) return TQP_ERR_ARG;
    if (!strcmp(name, "fuse_dgu")) {
        REQ(c, value == 0 || value == 1, TQP_ERR_ARG, "fuse_dgu must be 0 or 1");
        c->fuse_dgu = value;
        return TQP_OK;
    }
    if (!strcmp(name, "route_impl")) {
        REQ(c, value >= 0 && value <= 3, TQP_ERR_ARG, "route_impl must be 0..3");
        c->route_impl = value;
        return TQP_OK;
    }
    if (!strcmp(name, "gemm_impl")) {
        REQ(c, value >= 0 && value <= 3, TQP_ERR_ARG, "gemm_impl must be 0..3");
        c->gemm_impl = value;
        return TQP_OK;
    }
#ifdef TQP_TRACE   // instrumented builds only (see common.cuh)
    if (!strcmp(name, "trace")) {
        c->trace = value;
        c->trace_seq = 0;
        return TQP_OK;
    }
    if (!strcmp(name, "ablate")) {
        c->ablate = value;
        return TQP_OK;
    }
#endif
    if (!strcmp(name, "host_chunks")) {
        REQ(c, value == 0 || value == 1 || value == 4, TQP_ERR_ARG, "host_chunks must be 0 (auto), 1 or 4");
        c->host_chunks = value;
        return TQP_OK;
    }
    if (!strcmp(name, "time_gemm")) {
        c->time_gemm = value ? 1 : 0;
        if (value && c->ev.empty()) {
            c->ev.resize(8192);
            for (auto &e : c->ev) TQP_CUDA_OK(c, cudaEventCreate(&e));
        }
        c->ev_used = 0;
        return TQP_OK;
    }
    c->err = "unknown option";
    return TQP_ERR_ARG;
}

tqp_status tqp_route(tqp_ctx *c, int T, const void *X, const float *W_r, const float *logit_bias, int32_t *topk_idx,
                     float *topk_w, float *logits_out, void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, X); PTR_OK(c, W_r); PTR_OK(c, topk_idx); PTR_OK(c, topk_w);
    if (!logits_out && c->route_impl != 1 && route_screen_applicable(c, T, c->route_impl >= 2) && ((uintptr_t)X & 15) == 0) {
        CUtensorMap mx, mw;
        st = act_map(c, &mx, X, (uint64_t)T, c->desc.d, 128);
        if (st == TQP_OK) st = act_map(c, &mw, c->p<bf16>(c->ws.WrHL), (uint64_t)c->desc.E, 2 * (uint64_t)c->desc.d, 256);
        if (st != TQP_OK) return st;
        c->last_route_screened = 1;
        return launch_route_screened(c, T, (const bf16 *)X, W_r, logit_bias, topk_idx, topk_w, nullptr, &mx, &mw, (cudaStream_t)stream);
    }
    c->last_route_screened = 0;
    float *lg = logits_out ? logits_out : c->p<float>(c->ws.logits);
    return launch_route(c, T, (const bf16 *)X, W_r, logit_bias, topk_idx, topk_w, lg, (cudaStream_t)stream);
}

tqp_status tqp_route_info(tqp_ctx *c, int *screened, int *fallback, void *stream) {
    if (!c) return TQP_ERR_ARG;
    REQ(c, c->base != nullptr, TQP_ERR_WORKSPACE, "no workspace bound");
    if (screened) *screened = c->last_route_screened;
    if (fallback) {
        *fallback = 0;
        if (c->last_route_screened) {
            TQP_CUDA_OK(c, cudaMemcpyAsync(fallback, c->p<int>(c->ws.rflag), sizeof(int), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
            TQP_CUDA_OK(c, cudaStreamSynchronize((cudaStream_t)stream));
        }
    }
    return TQP_OK;
}

tqp_status tqp_dispatch(tqp_ctx *c, int T, const int32_t *topk_idx, int32_t *counts, int32_t *offsets, int32_t *perm,
                        int32_t *inv_perm, void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, topk_idx); PTR_OK(c, counts); PTR_OK(c, offsets); PTR_OK(c, perm); PTR_OK(c, inv_perm);
    c->disp_T = T;
    c->fwd_T = -1;
    c->zd_src = nullptr;
    return launch_dispatch(c, T, topk_idx, counts, offsets, perm, inv_perm, (cudaStream_t)stream);
}

tqp_status tqp_expert_fwd(tqp_ctx *c, int T, const void *X, const int32_t *offsets, const int32_t *perm, void *Ye,
                          void *stream) {
    tqp_status st = common_checks(c, T, true);
    if (st != TQP_OK) return st;
    PTR_OK(c, X); PTR_OK(c, offsets); PTR_OK(c, perm); PTR_OK(c, Ye);
    REQ(c, c->disp_T == T, TQP_ERR_STATE, "tqp_expert_fwd must follow tqp_dispatch with the same T");
    cudaStream_t s = (cudaStream_t)stream;
    const tqp_layer_desc &D = c->desc;
    const int N = T * D.k;
    const float ls = D.lora_scale;
    bf16 *Xp = c->p<bf16>(c->ws.Xp), *G = c->p<bf16>(c->ws.G), *U = c->p<bf16>(c->ws.U), *H = c->p<bf16>(c->ws.H);
#define CK(x) do { st = (x); if (st != TQP_OK) return st; } while (0)
    const bool fused = D.r == 16 || D.r == 32;   // rank 8 (config 0) keeps the separate CUDA-core kernels
    const bool tq = c->tq.on;
    if (tq) {
        // TurboQuant base: carry the adapters' input sides and the token rows into the rotated spaces once;
        // everything below then runs on x' = R_d x and A' = R A  (x . A = x' . A', x . W_row = norm level[codes] . x')
        CK(tq_rotate_adapter(c, &c->tq.w.space_d, (const bf16 *)c->tq.w.A_gate, c->tq.Ar_gate, s));
        CK(tq_rotate_adapter(c, &c->tq.w.space_d, (const bf16 *)c->tq.w.A_up, c->tq.Ar_up, s));
        CK(tq_rotate_adapter(c, &c->tq.w.space_F, (const bf16 *)c->tq.w.A_down, c->tq.Ar_down, s));
        CK(launch_tq_rotate(c, &c->tq.w.space_d, X, false, T, c->tq.Xr, false, 0, s));
        X = c->tq.Xr;
    }
    if (fused) {   // Xp = gather(X) and both adapter projections x.A_g | x.A_u in one pass over the rows
        if (D.d % 256 == 0) {   // rows by TMA gather4 (X is the caller's: its maps are encoded per call)
            CUtensorMap gm[3];
            CK(gather_maps(c, gm, X, (uint64_t)T, Xp, (uint64_t)N, D.d));
            CK(launch_rows_gather_proj(c, &gm[0], T, &gm[1], &gm[2], N, D.d, perm, nullptr, (const bf16 *)c->w.A_gate,
                                       (const bf16 *)c->w.A_up, 1, ls, c->p<bf16>(c->ws.XAg), c->p<bf16>(c->ws.XAu), s));
        } else {
            CK(launch_rows_proj(c, (const bf16 *)X, D.d, perm, nullptr, Xp, (const bf16 *)c->w.A_gate, (const bf16 *)c->w.A_up, 1,
                                ls, c->p<bf16>(c->ws.XAg), c->p<bf16>(c->ws.XAu), s));
        }
    } else {
        CK(launch_gather_rows(c, N, (const bf16 *)X, perm, Xp, s));
        CK(launch_rows_proj(c, Xp, D.d, nullptr, nullptr, nullptr, (const bf16 *)c->w.A_gate, (const bf16 *)c->w.A_up, 1, ls,
                            c->p<bf16>(c->ws.XAg), c->p<bf16>(c->ws.XAu), s));
    }
    GemmProblem pr[2] = {c->prob_gate, c->prob_up};
    CK(run_gemm(c, pr, 2, s));
    if (tq && c->tq.w.space_F.hadamard) {   // h' = R_F (silu(g) u) in one pass: h itself is never stored
        CK(launch_tq_swiglu_fwd_rot(c, &c->tq.w.space_F, G, U, H, N, s));
    } else {
        CK(launch_swiglu_fwd(c, N, G, U, H, s));
    }
    if (tq) {   // a dense R_F goes through the idle dG buffer
        if (!c->tq.w.space_F.hadamard) {
            CK(launch_tq_rotate(c, &c->tq.w.space_F, H, false, N, c->p<bf16>(c->ws.dG), false, 0, s));
            TQP_CUDA_OK(c, cudaMemcpyAsync(H, c->p<bf16>(c->ws.dG), (size_t)N * D.F * 2, cudaMemcpyDeviceToDevice, s));
        }
    }
    if (fused) CK(launch_rows_proj_tma(c, &c->prob_down.seg[0].act_map2, D.F, (const bf16 *)c->w.A_down, 1, ls, c->p<bf16>(c->ws.HAd), s));
    else CK(launch_rows_proj(c, H, D.F, nullptr, nullptr, nullptr, (const bf16 *)c->w.A_down, nullptr, 1, ls,
                             c->p<bf16>(c->ws.HAd), nullptr, s));
    GemmProblem pd = c->prob_down;
    pd.out = (bf16 *)Ye;
    CK(run_gemm(c, &pd, 1, s));
#undef CK
    c->fwd_T = D.training ? T : -1;
    return TQP_OK;
}

tqp_status tqp_combine(tqp_ctx *c, int T, const void *Ye, const int32_t *inv_perm, const float *topk_w, void *Y,
                       void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, Ye); PTR_OK(c, inv_perm); PTR_OK(c, topk_w); PTR_OK(c, Y);
    return launch_combine(c, T, (const bf16 *)Ye, inv_perm, topk_w, (bf16 *)Y, (cudaStream_t)stream);
}

tqp_status tqp_combine_bwd(tqp_ctx *c, int T, const void *dY, const void *Ye, const int32_t *inv_perm, const int32_t *perm,
                           const float *topk_w, void *dYe, float *dtopk_w, void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, dY); PTR_OK(c, inv_perm); PTR_OK(c, topk_w); PTR_OK(c, dYe);
    if (dtopk_w) PTR_OK(c, Ye);
    if (perm) REQ(c, aligned16(perm), TQP_ERR_ALIGN, "perm is not 16-byte aligned");
    const tqp_layer_desc &D = c->desc;
    c->zd_src = nullptr;
    if (perm && (D.r == 16 || D.r == 32) && D.training && c->have_weights) {
        // Fused: dYe[p] = w[a] dY[t] by sorted position (a = perm[p]) and, from the same rows, Zd = s dYe . B_d^T, the
        // adapter projection tqp_expert_bwd needs.  dw = <dY, Ye> is a separate reduction when asked for.
        if (D.d % 256 == 0) {
            CUtensorMap gm[3];
            st = gather_maps(c, gm, dY, (uint64_t)T, dYe, (uint64_t)T * D.k, D.d);
            if (st == TQP_OK)
                st = launch_rows_gather_proj(c, &gm[0], T, &gm[1], &gm[2], T * D.k, D.d, perm, topk_w, (const bf16 *)c->w.B_down,
                                             nullptr, 0, D.lora_scale, c->p<bf16>(c->ws.Zd), nullptr, (cudaStream_t)stream);
        } else {
            st = launch_rows_proj(c, (const bf16 *)dY, D.d, perm, topk_w, (bf16 *)dYe, (const bf16 *)c->w.B_down, nullptr, 0,
                                  D.lora_scale, c->p<bf16>(c->ws.Zd), nullptr, (cudaStream_t)stream);
        }
        if (st != TQP_OK) return st;
        c->zd_src = dYe;
        if (dtopk_w) st = launch_combine_dw(c, T, (const bf16 *)dY, (const bf16 *)Ye, inv_perm, dtopk_w, (cudaStream_t)stream);
        return st;
    }
    return launch_combine_bwd(c, T, (const bf16 *)dY, (const bf16 *)Ye, inv_perm, topk_w, (bf16 *)dYe, dtopk_w,
                              (cudaStream_t)stream);
}


tqp_status tqp_expert_bwd(tqp_ctx *c, int T, const void *X, const void *dYe, const int32_t *offsets, const int32_t *perm,
                          void *dXp, float *dA_gate, float *dB_gate, float *dA_up, float *dB_up, float *dA_down,
                          float *dB_down, int flags, void *stream) {
    tqp_status st = common_checks(c, T, true);
    if (st != TQP_OK) return st;
    PTR_OK(c, X); PTR_OK(c, dYe); PTR_OK(c, offsets); PTR_OK(c, perm); PTR_OK(c, dXp);
    PTR_OK(c, dA_gate); PTR_OK(c, dB_gate); PTR_OK(c, dA_up); PTR_OK(c, dB_up); PTR_OK(c, dA_down); PTR_OK(c, dB_down);
    REQ(c, c->desc.training == 1, TQP_ERR_STATE, "tqp_expert_bwd needs a ctx created with training=1");
    REQ(c, c->fwd_T == T, TQP_ERR_STATE, "tqp_expert_bwd must follow a training-mode tqp_expert_fwd with the same T");
    cudaStream_t s = (cudaStream_t)stream;
    const tqp_layer_desc &D = c->desc;
    const int N = T * D.k;
    const float ls = D.lora_scale;
    const bf16 *dye = (const bf16 *)dYe;
    bf16 *Xp = c->p<bf16>(c->ws.Xp), *G = c->p<bf16>(c->ws.G), *U = c->p<bf16>(c->ws.U), *H = c->p<bf16>(c->ws.H);
    bf16 *dH = c->p<bf16>(c->ws.dH), *dG = c->p<bf16>(c->ws.dG), *dU = c->p<bf16>(c->ws.dU);
    bf16 *Zd = c->p<bf16>(c->ws.Zd), *Zg = c->p<bf16>(c->ws.Zg), *Zu = c->p<bf16>(c->ws.Zu);
#define CK(x) do { st = (x); if (st != TQP_OK) return st; } while (0)
    REQ(c, (flags & ~TQP_BWD_DYE_UNMODIFIED) == 0, TQP_ERR_ARG, "unknown flag");
    if (flags & TQP_BWD_DYE_UNMODIFIED)
        REQ(c, c->zd_src == dYe, TQP_ERR_STATE,
            "TQP_BWD_DYE_UNMODIFIED: dYe is not the tensor the directly preceding fused tqp_combine_bwd (perm given) wrote");
    // down projection: dH = dYe . Wd_eff^T,  dB_d = (s h A_d)^T dYe,  dA_d = h^T (s dYe B_d^T)
    if (!(flags & TQP_BWD_DYE_UNMODIFIED))   // the caller does not vouch for the projection tqp_combine_bwd may have left
        CK(launch_rows_proj(c, dye, D.d, nullptr, nullptr, nullptr, (const bf16 *)c->w.B_down, nullptr, 0, ls, Zd, nullptr, s));
    c->zd_src = nullptr;
    GemmProblem ph = c->prob_dh;
    ph.seg[0].act = dye;
    CK(act_map(c, &ph.seg[0].act_map, dye, (uint64_t)N, D.d));
    CK(act_map(c, &ph.seg[0].act_map2, dye, (uint64_t)N, D.d, kTileRows / 2));
    CK(run_gemm(c, &ph, 1, s));
    const bool tq = c->tq.on;
    if (tq && c->tq.w.space_F.hadamard) {   // the GEMM produced dh' = R_F dh: un-rotate and apply the SwiGLU backward in one pass
        CK(launch_tq_swiglu_bwd_rot(c, &c->tq.w.space_F, dH, G, U, dG, dU, N, s));
    } else {
        if (tq) {
            CK(launch_tq_rotate(c, &c->tq.w.space_F, dH, false, N, dG, false, 1, s));
            TQP_CUDA_OK(c, cudaMemcpyAsync(dH, dG, (size_t)N * D.F * 2, cudaMemcpyDeviceToDevice, s));
        }
        CK(launch_swiglu_bwd(c, N, dH, G, U, dG, dU, s));
    }
    // With a TurboQuant base the dA gradients are first formed w.r.t. A' = R A (the rows that multiply them are rotated) and
    // then carried back, dA = R^T dA'; the deferred tail of tqp_step_host is not used in that mode.
    const bool defer = c->defer_tail && !tq;
    float *dAd = tq ? c->tq.dAr_down : dA_down, *dAg = tq ? c->tq.dAr_gate : dA_gate, *dAu = tq ? c->tq.dAr_up : dA_up;
    if (!defer) {
        CK(launch_rows_wgrad(c, dye, D.d, c->p<bf16>(c->ws.HAd), nullptr, offsets, 0, dB_down, nullptr, s));
        CK(launch_rows_wgrad(c, H, D.F, Zd, nullptr, offsets, 1, dAd, nullptr, s));
        if (tq) CK(tq_unrotate_grad(c, &c->tq.w.space_F, dAd, dA_down, s));
    }
    // gate / up projections: dXp = dG . Wg_eff^T + dU . Wu_eff^T and their adapter gradients
    // one pass over dG / dU for projection + dB (cfg 2: 189 -> 116 us; cfg 4, two tiles per expert and r = 32: 380 -> 335 us)
    const bool dgu = (D.r == 16 || D.r == 32) && c->fuse_dgu != 0;
    if (dgu) {   // projections and dB_gate / dB_up from one pass over dG and dU
        CK(launch_rows_proj_wgrad(c, &c->prob_dx.seg[0].act_map, &c->prob_dx.seg[1].act_map, D.F, (const bf16 *)c->w.B_gate, (const bf16 *)c->w.B_up,
                                  c->p<bf16>(c->ws.XAg), c->p<bf16>(c->ws.XAu), ls, Zg, Zu, dB_gate, dB_up, s));
    } else if (D.r == 16 || D.r == 32) {   // dG, dU are workspace tensors the dXp GEMM already has tensor maps for
        CK(launch_rows_proj_tma(c, &c->prob_dx.seg[0].act_map2, D.F, (const bf16 *)c->w.B_gate, 0, ls, Zg, s));
        CK(launch_rows_proj_tma(c, &c->prob_dx.seg[1].act_map2, D.F, (const bf16 *)c->w.B_up, 0, ls, Zu, s));
    } else {
        CK(launch_rows_proj(c, dG, D.F, nullptr, nullptr, nullptr, (const bf16 *)c->w.B_gate, nullptr, 0, ls, Zg, nullptr, s));
        CK(launch_rows_proj(c, dU, D.F, nullptr, nullptr, nullptr, (const bf16 *)c->w.B_up, nullptr, 0, ls, Zu, nullptr, s));
    }
    GemmProblem px = c->prob_dx;
    px.out = (bf16 *)dXp;
    CK(run_gemm(c, &px, 1, s));
    if (defer) {   // tqp_step_host: dX leaves for the host first (nothing below feeds it)
        c->tail = {dA_gate, dB_gate, dA_up, dB_up, dA_down, dB_down, dye, offsets, true, dgu};
        return TQP_OK;
    }
    if (!dgu) {
        CK(launch_rows_wgrad(c, dG, D.F, c->p<bf16>(c->ws.XAg), nullptr, offsets, 0, dB_gate, nullptr, s));
        CK(launch_rows_wgrad(c, dU, D.F, c->p<bf16>(c->ws.XAu), nullptr, offsets, 0, dB_up, nullptr, s));
    }
    CK(launch_rows_wgrad(c, Xp, D.d, Zg, Zu, offsets, 1, dAg, dAu, s));   // one pass over Xp for both
    if (tq) {
        CK(tq_unrotate_grad(c, &c->tq.w.space_d, dAg, dA_gate, s));
        CK(tq_unrotate_grad(c, &c->tq.w.space_d, dAu, dA_up, s));
    }
#undef CK
    return TQP_OK;
}

// the adapter weight gradients that tqp_expert_bwd left pending (defer_tail)
static tqp_status expert_bwd_tail(tqp_ctx *c, cudaStream_t s) {
    if (!c->tail.pending) return TQP_OK;
    c->tail.pending = false;
    c->launches = 0;
    const tqp_layer_desc &D = c->desc;
    tqp_status st;
#define CK(x) do { st = (x); if (st != TQP_OK) return st; } while (0)
    CK(launch_rows_wgrad(c, c->tail.dYe, D.d, c->p<bf16>(c->ws.HAd), nullptr, c->tail.offsets, 0, c->tail.dB_down, nullptr, s));
    CK(launch_rows_wgrad(c, c->p<bf16>(c->ws.H), D.F, c->p<bf16>(c->ws.Zd), nullptr, c->tail.offsets, 1, c->tail.dA_down, nullptr, s));
    if (!c->tail.dgu_done) {
        CK(launch_rows_wgrad(c, c->p<bf16>(c->ws.dG), D.F, c->p<bf16>(c->ws.XAg), nullptr, c->tail.offsets, 0, c->tail.dB_gate, nullptr, s));
        CK(launch_rows_wgrad(c, c->p<bf16>(c->ws.dU), D.F, c->p<bf16>(c->ws.XAu), nullptr, c->tail.offsets, 0, c->tail.dB_up, nullptr, s));
    }
    CK(launch_rows_wgrad(c, c->p<bf16>(c->ws.Xp), D.d, c->p<bf16>(c->ws.Zg), c->p<bf16>(c->ws.Zu), c->tail.offsets, 1, c->tail.dA_gate,
                         c->tail.dA_up, s));
#undef CK
    return TQP_OK;
}

tqp_status tqp_dispatch_bwd(tqp_ctx *c, int T, const void *dXp, const int32_t *inv_perm, void *dX, void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, dXp); PTR_OK(c, inv_perm); PTR_OK(c, dX);
    if (c->tq.on) {   // dXp is in the rotated input space: sum the tokens' rows there, then dX = R_d^T (sum)
        st = launch_combine(c, T, (const bf16 *)dXp, inv_perm, nullptr, c->tq.Xr, (cudaStream_t)stream);
        const int n1 = c->launches;
        if (st == TQP_OK) st = launch_tq_rotate(c, &c->tq.w.space_d, c->tq.Xr, false, T, dX, false, 1, (cudaStream_t)stream);
        (void)n1;
        return st;
    }
    return launch_combine(c, T, (const bf16 *)dXp, inv_perm, nullptr, (bf16 *)dX, (cudaStream_t)stream);
}

tqp_status tqp_route_bwd(tqp_ctx *c, int T, const void *X, const float *W_r, const int32_t *topk_idx,
                         const float *topk_w, const float *dtopk_w, const int32_t *offsets, const int32_t *perm, void *dX,
                         float *dW_r, void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, X); PTR_OK(c, W_r); PTR_OK(c, topk_idx); PTR_OK(c, topk_w); PTR_OK(c, dtopk_w); PTR_OK(c, offsets);
    PTR_OK(c, perm); PTR_OK(c, dX); PTR_OK(c, dW_r);
    return launch_route_bwd(c, T, (const bf16 *)X, W_r, topk_idx, topk_w, nullptr, dtopk_w, offsets, perm, (bf16 *)dX, dW_r,
                            (cudaStream_t)stream);
}

tqp_status tqp_route_sigmoid(tqp_ctx *c, int T, const void *X, const float *W_r, const float *select_bias, int32_t *topk_idx,
                             float *topk_w, float *topk_s, float *logits_out, void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, X); PTR_OK(c, W_r); PTR_OK(c, topk_idx); PTR_OK(c, topk_w); PTR_OK(c, topk_s);
    if (!logits_out && c->route_impl != 1 && route_screen_applicable(c, T, c->route_impl >= 2) && ((uintptr_t)X & 15) == 0) {
        CUtensorMap mx, mw;
        st = act_map(c, &mx, X, (uint64_t)T, c->desc.d, 128);
        if (st == TQP_OK) st = act_map(c, &mw, c->p<bf16>(c->ws.WrHL), (uint64_t)c->desc.E, 2 * (uint64_t)c->desc.d, 256);
        if (st != TQP_OK) return st;
        c->last_route_screened = 1;
        return launch_route_screened(c, T, (const bf16 *)X, W_r, select_bias, topk_idx, topk_w, topk_s, &mx, &mw, (cudaStream_t)stream);
    }
    c->last_route_screened = 0;
    float *lg = logits_out ? logits_out : c->p<float>(c->ws.logits);
    return launch_route_sigmoid(c, T, (const bf16 *)X, W_r, select_bias, topk_idx, topk_w, topk_s, lg, (cudaStream_t)stream);
}

tqp_status tqp_route_sigmoid_bwd(tqp_ctx *c, int T, const void *X, const float *W_r, const int32_t *topk_idx,
                                 const float *topk_w, const float *topk_s, const float *dtopk_w, const int32_t *offsets,
                                 const int32_t *perm, void *dX, float *dW_r, void *stream) {
    tqp_status st = common_checks(c, T, false);
    if (st != TQP_OK) return st;
    PTR_OK(c, X); PTR_OK(c, W_r); PTR_OK(c, topk_idx); PTR_OK(c, topk_w); PTR_OK(c, topk_s); PTR_OK(c, dtopk_w);
    PTR_OK(c, offsets); PTR_OK(c, perm); PTR_OK(c, dX); PTR_OK(c, dW_r);
    return launch_route_bwd(c, T, (const bf16 *)X, W_r, topk_idx, topk_w, topk_s, dtopk_w, offsets, perm, (bf16 *)dX, dW_r,
                            (cudaStream_t)stream);
}

tqp_status tqp_bias_update(tqp_ctx *c, const int32_t *counts, float *bias, int mode, float gamma, float cap_hi, float cap_lo,
                           void *stream) {
    if (!c) return TQP_ERR_ARG;
    c->launches = 0;
    PTR_OK(c, counts); PTR_OK(c, bias);
    REQ(c, mode == 0 || mode == 1, TQP_ERR_ARG, "mode must be 0 (sign-based) or 1 (three-tier)");
    REQ(c, mode == 0 || cap_hi > 0.f, TQP_ERR_ARG, "three-tier controller needs cap_hi > 0");
    return launch_bias_update(c, counts, bias, mode, gamma, cap_hi, cap_lo, (cudaStream_t)stream);
}

tqp_status tqp_consolidate(tqp_ctx *c, int pack, int e0, int n_experts, void *W_out, void *stream) {
    if (!c) return TQP_ERR_ARG;
    c->launches = 0;
    REQ(c, c->have_weights && !c->tq.on, TQP_ERR_STATE, "tqp_consolidate needs tqp_bind_weights (vector-quantised base) first");
    REQ(c, pack >= 0 && pack <= 2, TQP_ERR_ARG, "pack must be 0 (gate), 1 (up) or 2 (down)");
    REQ(c, e0 >= 0 && n_experts >= 0 && e0 + n_experts <= c->desc.E, TQP_ERR_ARG, "expert range outside [0, E)");
    if (n_experts == 0) return TQP_OK;
    PTR_OK(c, W_out);
    return launch_consolidate(c, pack, e0, n_experts, (bf16 *)W_out, (cudaStream_t)stream);
}

tqp_status tqp_step_host(tqp_ctx *c, int T, const void *X_host, const void *dY_host, const float *W_r,
                         const float *logit_bias, void *Y_host, void *dX_host, float *dA_gate, float *dB_gate,
                         float *dA_up, float *dB_up, float *dA_down, float *dB_down, float *dW_r, void *stream) {
    tqp_status st = tqp_step_host_async(c, T, X_host, dY_host, W_r, logit_bias, Y_host, dX_host, dA_gate, dB_gate, dA_up, dB_up,
                                        dA_down, dB_down, dW_r, stream);
    if (st != TQP_OK) return st;
    const int launches = c->launches;
    st = tqp_step_host_wait(c, 0);
    if (st != TQP_OK) return st;
    TQP_CUDA_OK(c, cudaStreamSynchronize((cudaStream_t)stream));
    c->launches = launches;
    return TQP_OK;
}

tqp_status tqp_step_host_wait(tqp_ctx *c, int age) {
    if (!c) return TQP_ERR_ARG;
    REQ(c, age == 0 || age == 1, TQP_ERR_ARG, "age must be 0 (latest step) or 1 (the one before)");
    const long long seq = c->host_seq - 1 - age;
    if (seq < 0 || !c->ev_done[0]) return TQP_OK;   // nothing that old is in flight
    TQP_CUDA_OK(c, cudaEventSynchronize(c->ev_done[seq & 1]));
    TQP_CUDA_OK(c, cudaEventSynchronize(c->ev_comp[seq & 1]));
    return TQP_OK;
}

tqp_status tqp_step_host_async(tqp_ctx *c, int T, const void *X_host, const void *dY_host, const float *W_r,
                               const float *logit_bias, void *Y_host, void *dX_host, float *dA_gate, float *dB_gate,
                               float *dA_up, float *dB_up, float *dA_down, float *dB_down, float *dW_r, void *stream) {
    tqp_status st = common_checks(c, T, true);
    if (st != TQP_OK) return st;
    REQ(c, X_host && dY_host && Y_host && dX_host, TQP_ERR_ARG, "host buffer is NULL");
    cudaStream_t s = (cudaStream_t)stream;
    const tqp_layer_desc &D = c->desc;
    const size_t row_bytes = (size_t)T * D.d * 2;
    const int par = (int)(c->host_seq & 1);   // upload staging set of this step
    if (!c->host_base) {   // first use: the library's own staging (freed by tqp_destroy)
        TQP_CUDA_OK(c, cudaMalloc(&c->host_base, c->ws.host_total));
        TQP_CUDA_OK(c, cudaMemsetAsync(c->host_base, 0, c->ws.host_total, s));
    }
    auto hp = [&](size_t off) { return c->host_base + off; };
    bf16 *X = (bf16 *)hp(par ? c->ws.hX2 : c->ws.hX), *dY = (bf16 *)hp(par ? c->ws.hdY2 : c->ws.hdY);
    bf16 *Y = (bf16 *)hp(c->ws.hY), *dX = (bf16 *)hp(c->ws.hdX);
    int32_t *ti = (int32_t *)hp(c->ws.topk_idx), *counts = (int32_t *)hp(c->ws.counts), *offs = (int32_t *)hp(c->ws.offsets);
    int32_t *perm = (int32_t *)hp(c->ws.perm), *inv = (int32_t *)hp(c->ws.inv_perm);
    float *tw = (float *)hp(c->ws.topk_w), *dtw = (float *)hp(c->ws.dtopk_w);
    bf16 *Ye = (bf16 *)hp(c->ws.Ye), *dYe = (bf16 *)hp(c->ws.dYe), *dXp = (bf16 *)hp(c->ws.dXp);
    int total = 0;
#define CK(x) do { st = (x); total += c->launches; if (st != TQP_OK) return st; } while (0)
    if (!c->copy_in) {
        TQP_CUDA_OK(c, cudaStreamCreateWithFlags(&c->copy_in, cudaStreamNonBlocking));
        TQP_CUDA_OK(c, cudaStreamCreateWithFlags(&c->copy_out, cudaStreamNonBlocking));
        for (cudaEvent_t *e : {&c->ev_start, &c->ev_x, &c->ev_dy, &c->ev_y, &c->ev_yout, &c->ev_dx, &c->ev_xc[0], &c->ev_xc[1],
                               &c->ev_xc[2], &c->ev_xc[3], &c->ev_done[0], &c->ev_done[1], &c->ev_comp[0], &c->ev_comp[1]})
            TQP_CUDA_OK(c, cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    }
    // X goes up in four token chunks and the router (token-wise) starts on each chunk as it lands; dY follows on the same
    // copy stream while the forward pass already runs on `s`; Y comes down on a second copy stream under the backward
    // pass (PCIe is full duplex); dX leaves before the last adapter weight gradients are computed.  The kernels are
    // ordered after what `s` held before.  The uploads are NOT: they only wait for the step before last, which used the
    // same staging set (its kernels read X until the end of its backward pass), so that the uploads of a step issued
    // while the previous one is still running travel under that step's kernels.
    if (c->host_seq >= 2) {
        TQP_CUDA_OK(c, cudaStreamWaitEvent(c->copy_in, c->ev_comp[par], 0));
    } else {   // first use of this staging set: order the uploads after what `s` holds now (e.g. tqp_bind_workspace's zero-fill)
        TQP_CUDA_OK(c, cudaEventRecord(c->ev_start, s));
        TQP_CUDA_OK(c, cudaStreamWaitEvent(c->copy_in, c->ev_start, 0));
    }
    {
        // With the previous step still running its kernels, this step's X will have landed long before `s` gets to the
        // router: upload and route it in one piece then (four router launches of T / 4 tokens fill the SMs worse than one).
        // (Which of the two is taken depends on timing; both give the same bits -- the router is token-wise -- and the option
        // "host_chunks" = 1 / 4 pins the choice for tests.)
        const bool behind = c->host_seq >= 1 && cudaEventQuery(c->ev_comp[par ^ 1]) == cudaErrorNotReady;
        const int nch = c->host_chunks ? c->host_chunks : (T >= 1024 && !behind) ? 4 : 1, per = ((T + nch - 1) / nch + 3) & ~3;   // chunk starts stay 16-byte aligned in every array
        for (int ch = 0; ch < nch; ++ch) {
            const int t0 = ch * per, tc = std::min(per, T - t0);
            if (tc <= 0) break;
            const size_t eo = (size_t)t0 * D.d;
            TQP_CUDA_OK(c, cudaMemcpyAsync(X + eo, (const bf16 *)X_host + eo, (size_t)tc * D.d * 2, cudaMemcpyHostToDevice, c->copy_in));
            TQP_CUDA_OK(c, cudaEventRecord(c->ev_xc[ch], c->copy_in));
            TQP_CUDA_OK(c, cudaStreamWaitEvent(s, c->ev_xc[ch], 0));
            CK(tqp_route(c, tc, X + eo, W_r, logit_bias, ti + (size_t)t0 * D.k, tw + (size_t)t0 * D.k, nullptr, s));
        }
    }
    TQP_CUDA_OK(c, cudaMemcpyAsync(dY, dY_host, row_bytes, cudaMemcpyHostToDevice, c->copy_in));
    TQP_CUDA_OK(c, cudaEventRecord(c->ev_dy, c->copy_in));
    CK(tqp_dispatch(c, T, ti, counts, offs, perm, inv, s));
    CK(tqp_expert_fwd(c, T, X, offs, perm, Ye, s));
    if (c->host_seq >= 1) TQP_CUDA_OK(c, cudaStreamWaitEvent(s, c->ev_done[par ^ 1], 0));   // the previous step's Y and dX have left
    CK(tqp_combine(c, T, Ye, inv, tw, Y, s));
    TQP_CUDA_OK(c, cudaEventRecord(c->ev_y, s));
    TQP_CUDA_OK(c, cudaStreamWaitEvent(c->copy_out, c->ev_y, 0));
    TQP_CUDA_OK(c, cudaMemcpyAsync(Y_host, Y, row_bytes, cudaMemcpyDeviceToHost, c->copy_out));
    TQP_CUDA_OK(c, cudaEventRecord(c->ev_yout, c->copy_out));
    TQP_CUDA_OK(c, cudaStreamWaitEvent(s, c->ev_dy, 0));
    CK(tqp_combine_bwd(c, T, dY, Ye, inv, perm, tw, dYe, dW_r ? dtw : nullptr, s));
    c->defer_tail = 1;
    st = tqp_expert_bwd(c, T, X, dYe, offs, perm, dXp, dA_gate, dB_gate, dA_up, dB_up, dA_down, dB_down,
                        c->zd_src == dYe ? TQP_BWD_DYE_UNMODIFIED : 0, s);
    c->defer_tail = 0;
    total += c->launches;
    if (st != TQP_OK) { c->tail.pending = false; return st; }
    CK(tqp_dispatch_bwd(c, T, dXp, inv, dX, s));
    if (dW_r) CK(tqp_route_bwd(c, T, X, W_r, ti, tw, dtw, offs, perm, dX, dW_r, s));
    TQP_CUDA_OK(c, cudaEventRecord(c->ev_dx, s));
    TQP_CUDA_OK(c, cudaStreamWaitEvent(c->copy_out, c->ev_dx, 0));   // after the Y download on the same copy stream
    TQP_CUDA_OK(c, cudaMemcpyAsync(dX_host, dX, row_bytes, cudaMemcpyDeviceToHost, c->copy_out));
    TQP_CUDA_OK(c, cudaEventRecord(c->ev_done[par], c->copy_out));
    CK(expert_bwd_tail(c, s));
#undef CK
    TQP_CUDA_OK(c, cudaEventRecord(c->ev_comp[par], s));
    ++c->host_seq;
    c->launches = total;
    return TQP_OK;
}

void *tqp_debug_buffer(tqp_ctx *c, const char *name) {
    if (!c || !name || !c->base) return nullptr;
    struct { const char *n; size_t off; } tab[] = {
        {"G", c->ws.G}, {"U", c->ws.U}, {"H", c->ws.H}, {"Xp", c->ws.Xp}, {"dH", c->ws.dH}, {"dG", c->ws.dG},
        {"dU", c->ws.dU}, {"num_tiles", c->ws.num_tiles}, {"tiles", c->ws.tiles}, {"XAg", c->ws.XAg}, {"Zd", c->ws.Zd},
        {"logits", c->ws.logits}, {"lut", c->ws.lut}, {"trace", c->ws.trace}};
    for (auto &t : tab)
        if (!strcmp(t.n, name)) return c->base + t.off;
    return nullptr;
}

int tqp_last_launch_count(const tqp_ctx *c) { return c ? c->launches : 0; }

const char *tqp_status_string(tqp_status s) {
    switch (s) {
        case TQP_OK: return "TQP_OK";
        case TQP_ERR_ARG: return "TQP_ERR_ARG";
        case TQP_ERR_SHAPE: return "TQP_ERR_SHAPE";
        case TQP_ERR_ALIGN: return "TQP_ERR_ALIGN";
        case TQP_ERR_WORKSPACE: return "TQP_ERR_WORKSPACE";
        case TQP_ERR_STATE: return "TQP_ERR_STATE";
        case TQP_ERR_ARCH: return "TQP_ERR_ARCH";
        case TQP_ERR_CUDA: return "TQP_ERR_CUDA";
    }
    return "TQP_ERR_UNKNOWN";
}

const char *tqp_last_error(const tqp_ctx *c) { return c ? c->err.c_str() : ""; }

}  // extern "C"
