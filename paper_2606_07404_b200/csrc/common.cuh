// Shared declarations of the TQP routed-expert library (sm_100a).  Product code: nothing here is shared
// with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <utility>
#include <vector>

#include "../../include/tqp.h"

namespace tqp {

typedef __nv_bfloat16 bf16;

// Debug instrumentation (clock64 timelines of one CTA pair, ablation switches that make results wrong on purpose) exists only
// in builds compiled with -DTQP_TRACE; in the product build TQP_DBG(x) is the constant 0 and the compiler drops those branches.
#ifdef TQP_TRACE
#define TQP_DBG(x) (x)
#else
#define TQP_DBG(x) 0
#endif

constexpr int kTileRows = 256;   // max routed rows (UMMA N) of one grouped-GEMM tile
constexpr int kRowPad = 512;     // rows of slack after N in every [N][*] workspace tensor (TMA boxes / 16-row groups over-read)
constexpr int kLoraPad = 64;     // adapter projections are stored [N][64] bf16 (one 128-byte swizzle row)
constexpr int kDispChunk = 256;  // assignments per warp in the dispatch kernels
constexpr int kWgradSeg = 512;   // rows per CTA of the adapter weight-gradient kernels; longer experts are split and reduced in order

struct Tile {          // one token tile of the grouped GEMMs: rows [row0, row0+rows) all belong to `expert`
    int32_t expert, row0, rows, pad;
};

// One GEMM "problem": out[p][m] = sum_seg sum_k act_seg[p][k] * Wdeq_seg[m][k] + sum_l lact_l[p][q] * lw_l[m][q]
// (swap-AB on the tensor cores: M = weight output channels, N = routed rows).
struct GemmSeg {
    const bf16 *act;        // [N][K] bf16 activations (B operand)
    const uint8_t *idx;     // codes of all experts
    const __half *scale;    // per-output-channel scales of all experts
    const uint32_t *scale2; // MN-major (backward) VQ segments: the scales as bf16 pairs (s, s), converted at bind time
    const float *norm;      // scalar (TurboQuant) format: fp32 row norms of all experts, in place of `scale`
    const void *lut;        // scalar format: the 256 bf16 Lloyd-Max levels of this pack's input space (device)
    int scalar;             // 1: TurboQuant codes, idx[e][M][K] / idx[e][K][M] one byte per weight; 0: vector-quantised
    int K;                  // contraction length of this segment
    int kmajor;             // 1: idx[e][M][K/8] (forward), 0: idx[e][K][M/8] (backward, transposed use)
    CUtensorMap act_map;    // box {64, kTileRows} over act, SWIZZLE_128B (1-CTA kernel)
    CUtensorMap act_map2;   // box {64, kTileRows/2}: one CTA's half of the rows (2-CTA kernel)
    CUtensorMap idx_map;    // box {16, 128} over idx viewed as [rows][bytes]
};
struct GemmLora {
    const bf16 *lact;       // [N][kLoraPad] bf16 (already multiplied by lora_scale)
    const bf16 *lw;         // adapter matrix of all experts
    int mk_layout;          // 1: lw[e][M][r] (K-major), 0: lw[e][r][M]
    CUtensorMap lact_map;   // box {64, kTileRows}
    CUtensorMap lact_map2;  // box {64, kTileRows/2}
};
struct GemmProblem {
    GemmSeg seg[2];
    GemmLora lora[2];
    int nseg, nlora;
    int M;                  // output channels
    int r;
    bf16 *out;              // [N][M]
};

struct GemmArgs {           // passed by value (__grid_constant__) so the tensor maps live in param space
    GemmProblem p[2];
    int nprob;
};

// derived device copies of a dense TurboQuant rotation (turboquant.cu), owned by the ctx
struct TqRot {
    const double *R;   // the caller's matrix (cache key)
    int n;
    bf16 *Rb, *Rtb;    // bf16 R and R^T (activation products)
    double *Rt;        // fp64 R^T
};

// TurboQuant-format layer state (tqp_bind_weights_tq): library-owned device buffers for the rotated activations / adapters
struct TqLayer {
    bool on = false;
    tqp_tq_weights w;
    bf16 *Xr = nullptr;                                    // [T_max][d] rotated X; reused for the rotated dX before it is turned back
    bf16 *Ar_gate = nullptr, *Ar_up = nullptr, *Ar_down = nullptr;   // R A: the adapters' input side in the rotated space
    bf16 *tmp_a = nullptr, *tmp_b = nullptr;               // [E][r][max(d,F)] transposition scratch
    float *dAr_gate = nullptr, *dAr_up = nullptr, *dAr_down = nullptr, *tmp_f = nullptr;   // gradients w.r.t. R A, fp32
    bf16 *lut_d = nullptr, *lut_F = nullptr;               // the 256 Lloyd-Max levels of either space as bf16
};

struct Workspace {
    // sizes
    size_t total = 0;        // the caller's workspace
    size_t host_total = 0;   // tqp_step_host staging (library-owned, allocated on first use)
    // offsets (bytes) into the bound buffer
    size_t Xp, G, U, H, dH, dG, dU, XAg, XAu, HAd, Zd, Zg, Zu, logits, blk_counts, tiles, num_tiles, xsegs, xfirst, tfirst, wg_scratch, wg_done, sched, lut, sc2, WrT, WrHL, wnorm, rflag, dl,
        // tqp_step_host staging
        trace, hX, hdY, hX2, hdY2, hY, hdX, topk_idx, topk_w, counts, offsets, perm, inv_perm, Ye, dYe, dXp, dtopk_w;
};

}  // namespace tqp

struct tqp_ctx {
    tqp_layer_desc desc;
    tqp::Workspace ws;
    char *base = nullptr;       // bound workspace
    char *host_base = nullptr;  // tqp_step_host staging (cudaMalloc on first use)
    size_t bound_bytes = 0;
    tqp_weights w;
    bool have_weights = false;
    int last_route_screened = 0;
    int route_impl = 0;         // 0 screened router where it pays, 1 dense exact chain, 2 screened wherever applicable, 3 = 2 with the self-check forced to fail
    int gemm_impl = 0;          // 0 tcgen05 CTA-pair kernel, 1 scaffold, 2 tcgen05 single-CTA kernel
    int fwd_T = -1;             // T of the last training-mode expert_fwd (TQP_ERR_STATE check)
    int disp_T = -1;
    // Set by the fused tqp_combine_bwd: ws.Zd holds s dYe.B_d^T of the dYe tensor it wrote (kept only to VALIDATE the caller's
    // TQP_BWD_DYE_UNMODIFIED claim in tqp_expert_bwd, never dereferenced); cleared by every other call that could invalidate it
    const void *zd_src = nullptr;
    int device = 0;                 // the device the ctx was created on (kernel attributes are per device)
    std::vector<tqp::TqRot> tq_rots;             // library-owned; freed by tqp_destroy
    tqp::TqLayer tq;                             // TurboQuant-format weights bound (tqp_bind_weights_tq)
    std::vector<std::pair<const void *, int>> smem_attr_done;   // kernels whose dynamic shared-memory limit has been raised on `device`, and to what
    int launches = 0;
    int num_sms = 148;
    int max_tiles = 0;
    int max_xsegs = 0;          // upper bound of the extra weight-gradient segments (N / kWgradSeg)
    std::string err;
    int ablate = 0;             // timing experiments only (tqp_set_option "ablate")
    int trace = 0;              // debug: n > 0 records a clock64 timeline of one cluster in the n-th CTA-pair GEMM launch from now
    int trace_seq = 0;
    int time_gemm = 0;          // bracket GEMM launches with events (tqp_gemm_time)
    // tqp_step_host: copy streams + events so that dY uploads and Y downloads overlap the compute on `stream`
    cudaStream_t copy_in = nullptr, copy_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_x = nullptr, ev_dy = nullptr, ev_y = nullptr, ev_yout = nullptr, ev_dx = nullptr;
    cudaEvent_t ev_xc[4] = {nullptr, nullptr, nullptr, nullptr};   // X arrives in token chunks; the router starts on the first
    // tqp_step_host_async: steps alternate between two upload staging sets so that the next step's X / dY travel while this
    // step computes; ev_done[p] = the step that used set p has delivered Y and dX to the host, ev_comp[p] = its kernels are done
    cudaEvent_t ev_done[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr};
    long long host_seq = 0;
    int host_chunks = 0;        // tqp_step_host_async: X upload / router in 1 or 4 token chunks (0: chosen at run time)
    // tqp_step_host defers all adapter weight gradients (nothing else depends on them) until dX is on its way to the host
    int defer_tail = 0;
    int fuse_dgu = 1;           // dG / dU: adapter projection and dB in one pass (rows_proj_wgrad_kernel) for r = 16 / 32; 0 = separate passes
    struct { float *dA_gate, *dB_gate, *dA_up, *dB_up, *dA_down, *dB_down; const tqp::bf16 *dYe; const int32_t *offsets; bool pending; bool dgu_done; } tail = {};
    std::vector<cudaEvent_t> ev; // pairs (start, stop)
    int ev_used = 0;
    // tensor maps over weights / workspace (built in bind_weights)
    tqp::GemmProblem prob_gate, prob_up, prob_down, prob_dh, prob_dx;

    template <class T> T *p(size_t off) const { return reinterpret_cast<T *>(base + off); }
};

namespace tqp {

#define TQP_CUDA_OK(ctx, call)                                                          \
    do {                                                                                \
        cudaError_t e__ = (call);                                                       \
        if (e__ != cudaSuccess) {                                                       \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);           \
            return TQP_ERR_CUDA;                                                        \
        }                                                                               \
    } while (0)

#define TQP_LAUNCH_OK(ctx)                                                              \
    do {                                                                                \
        (ctx)->launches++;                                                              \
        cudaError_t e__ = cudaGetLastError();                                           \
        if (e__ != cudaSuccess) {                                                       \
            (ctx)->err = std::string(__FILE__) + ":" + std::to_string(__LINE__) + ": " + cudaGetErrorString(e__); \
            return TQP_ERR_CUDA;                                                        \
        }                                                                               \
    } while (0)

// ---- kernels.cu ----------------------------------------------------------------------------------------
// gate (device int, or NULL): when given, both kernels return at once unless *gate != 0
tqp_status launch_route(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *bias, int32_t *topk_idx,
                        float *topk_w, float *logits, cudaStream_t s, const int *gate = nullptr);
// Screened router (route.cu): same results as launch_route, bit for bit; mapX = X as bf16 [T][d], box {64, 128}, mapW = the
// bf16 hi|lo split of W_r^T in the workspace [E][2d], box {64, 256}, both SWIZZLE_128B.
bool route_screen_applicable(const tqp_ctx *c, int T, bool forced);
tqp_status launch_route_screened(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *bias, int32_t *topk_idx,
                                 float *topk_w, float *topk_s /* non-NULL: sigmoid variant */, const CUtensorMap *mapX,
                                 const CUtensorMap *mapW, cudaStream_t s);
tqp_status launch_dispatch(tqp_ctx *c, int T, const int32_t *topk_idx, int32_t *counts, int32_t *offsets,
                           int32_t *perm, int32_t *inv_perm, cudaStream_t s);
tqp_status launch_gather_rows(tqp_ctx *c, int N, const bf16 *X, const int32_t *perm, bf16 *Xp, cudaStream_t s);
tqp_status launch_swiglu_fwd(tqp_ctx *c, int N, const bf16 *G, const bf16 *U, bf16 *H, cudaStream_t s);
tqp_status launch_swiglu_bwd(tqp_ctx *c, int N, const bf16 *dH, const bf16 *G, const bf16 *U, bf16 *dG, bf16 *dU,
                             cudaStream_t s);
tqp_status launch_combine(tqp_ctx *c, int T, const bf16 *Ye, const int32_t *inv_perm, const float *topk_w, bf16 *Y,
                          cudaStream_t s);
tqp_status launch_combine_bwd(tqp_ctx *c, int T, const bf16 *dY, const bf16 *Ye, const int32_t *inv_perm,
                              const float *topk_w, bf16 *dYe, float *dtopk_w, cudaStream_t s);
tqp_status launch_route_bwd(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const int32_t *topk_idx,
                            const float *topk_w, const float *topk_s, const float *dtopk_w, const int32_t *offsets,
                            const int32_t *perm, bf16 *dX, float *dW_r, cudaStream_t s);
tqp_status launch_route_sigmoid(tqp_ctx *c, int T, const bf16 *X, const float *W_r, const float *select_bias, int32_t *topk_idx,
                                float *topk_w, float *topk_s, float *logits, cudaStream_t s, const int *gate = nullptr);
tqp_status launch_bias_update(tqp_ctx *c, const int32_t *counts, float *bias, int mode, float gamma, float cap_hi, float cap_lo,
                              cudaStream_t s);
tqp_status launch_combine_dw(tqp_ctx *c, int T, const bf16 *dY, const bf16 *Ye, const int32_t *inv_perm, float *dtopk_w,
                             cudaStream_t s);
tqp_status launch_make_lut(tqp_ctx *c, const __half *codebook, bf16 *lut, cudaStream_t s);
tqp_status launch_scale_pairs(tqp_ctx *c, const __half *scale, uint32_t *out, size_t n, cudaStream_t s);

// ---- lora.cu -------------------------------------------------------------------------------------------
// out_w[p][0..r) = s * row(p) . W_w[e]  for w < (W1 ? 2 : 1); W_e is [K][r] if w_kr else [r][K]; out is [N][kLoraPad] bf16.
// row(p) = in[p], or with perm: in[perm[p]/k] (* roww[perm[p]] rounded to bf16), also written to through[p][K] if given.
tqp_status launch_rows_proj(tqp_ctx *c, const bf16 *in, int K, const int32_t *perm, const float *roww, bf16 *through,
                            const bf16 *W0, const bf16 *W1, int w_kr, float s, bf16 *out0, bf16 *out1, cudaStream_t st);
// the same for ONE adapter matrix and a dense workspace tensor read through its GEMM tensor map (r = 16 / 32 only)
tqp_status launch_rows_proj_tma(tqp_ctx *c, const CUtensorMap *map, int K, const bf16 *W, int w_kr, float s, bf16 *out, cudaStream_t st);
// the gathered variants (perm != nullptr) with rows by TMA gather4 and the write-through by TMA store (lora.cu); needs
// K % 256 == 0 and r = 16 / 32; maps as built by gather_maps() in api.cu
tqp_status launch_rows_gather_proj(tqp_ctx *c, const CUtensorMap *in_map, int in_rows, const CUtensorMap *out_map, const CUtensorMap *sc_map,
                                   int out_rows, int K, const int32_t *perm, const float *roww, const bf16 *W0, const bf16 *W1, int w_kr,
                                   float s, bf16 *out0, bf16 *out1, cudaStream_t st);
// W[e - e0][out][in] = bf16(deq + s A B) for experts e0 .. e0 + n_experts of pack 0 (gate) / 1 (up) / 2 (down) (consolidate.cu)
tqp_status launch_consolidate(tqp_ctx *c, int pack, int e0, int n_experts, bf16 *W, cudaStream_t st);
// grad_w[e] = sum_{p in e} small_w[p][q] * big[p][a]; stored [a][q] (out_ar=1: dA) or [q][a] (out_ar=0: dB), fp32
tqp_status launch_rows_proj_wgrad(tqp_ctx *c, const CUtensorMap *map_g, const CUtensorMap *map_u, int F, const bf16 *B_gate, const bf16 *B_up,
                                  const bf16 *XAg, const bf16 *XAu, float s, bf16 *Zg, bf16 *Zu, float *dB_gate, float *dB_up, cudaStream_t st);
tqp_status launch_rows_wgrad(tqp_ctx *c, const bf16 *big, int width, const bf16 *small0, const bf16 *small1,
                             const int32_t *offsets, int out_ar, float *grad0, float *grad1, cudaStream_t st);

// ---- gemm_scaffold.cu / gemm_tcgen05.cu -----------------------------------------------------------------
tqp_status launch_gemm_scaffold(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st);
tqp_status launch_gemm_tcgen05(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st);       // 1 CTA / tile
tqp_status launch_gemm_tcgen05_2cta(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st);  // CTA pair / tile
tqp_status launch_gemm_tcgen05_ts2(tqp_ctx *c, const GemmProblem *probs, int nprob, cudaStream_t st);   // CTA pair, weight operand in TMEM, 128-wide A stages (default)

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: raised once per ctx (a ctx lives on one device)
inline tqp_status ensure_dyn_smem(tqp_ctx *c, const void *func, int bytes) {
    for (auto &f : c->smem_attr_done)
        if (f.first == func) {
            if (f.second >= bytes) return TQP_OK;
            cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);   // a larger request than before
            if (e != cudaSuccess) { c->err = std::string("cudaFuncSetAttribute(MaxDynamicSharedMemorySize): ") + cudaGetErrorString(e); return TQP_ERR_CUDA; }
            f.second = bytes;
            return TQP_OK;
        }
    cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) {
        c->err = std::string("cudaFuncSetAttribute(MaxDynamicSharedMemorySize): ") + cudaGetErrorString(e);
        return TQP_ERR_CUDA;
    }
    c->smem_attr_done.push_back({func, bytes});
    return TQP_OK;
}

// ---- turboquant.cu --------------------------------------------------------------------------------------
tqp_status tq_check_space(tqp_ctx *c, const tqp_tq_space *sp);
tqp_status launch_tq_rotate(tqp_ctx *c, const tqp_tq_space *sp, const void *X, bool in_f32, long long rows, void *Y, bool out_f32, int inverse,
                            cudaStream_t st);
tqp_status launch_tq_swiglu_fwd_rot(tqp_ctx *c, const tqp_tq_space *sp, const bf16 *G, const bf16 *U, bf16 *Hr, long long rows, cudaStream_t st);
tqp_status launch_tq_swiglu_bwd_rot(tqp_ctx *c, const tqp_tq_space *sp, const bf16 *dHr, const bf16 *G, const bf16 *U, bf16 *dG, bf16 *dU,
                                    long long rows, cudaStream_t st);
tqp_status launch_tq_make_lut(tqp_ctx *c, const double *levels, bf16 *lut, cudaStream_t st);
template <typename T>
tqp_status launch_tq_fwht_strided(tqp_ctx *c, const tqp_tq_space *sp, const T *X, T *Y, int E, int r, int inverse, cudaStream_t st);   // [E][n][r], FWHT over n
template <typename T>
tqp_status launch_tq_transpose(tqp_ctx *c, const T *in, T *out, int E, int a, int b, cudaStream_t st);   // [E][a][b] -> [E][b][a]

// ---- device helpers ------------------------------------------------------------------------------------
__device__ __forceinline__ float bf16_bits_to_float(uint16_t b) { return __uint_as_float(((uint32_t)b) << 16); }
__device__ __forceinline__ float2 bf16x2_to_float2(uint32_t v) {
    return make_float2(__uint_as_float(v << 16), __uint_as_float(v & 0xffff0000u));
}
__device__ __forceinline__ uint32_t float2_to_bf16x2(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&t);
}

}  // namespace tqp
