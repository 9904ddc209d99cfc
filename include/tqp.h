/* tqp.h — C ABI of the B200-native routed-expert layer of the TQP method
 * ("Reversible Foundations: Training a 120B Sparse MoE through State-Preserving Scaling", arxiv 2606.07404).
 *
 * The path (§3.4 L224 router; Table 4 L237-239 top-k routed experts; §5.1 L401 gate/up/down
 * projections; §9.1 L938 rank-r adapters on each of the three packs, frozen base; §9.2 "reconstruction
 * looks up the codebook values and rescales by the stored norm"):
 *
 *   forward :  tqp_route -> tqp_dispatch -> tqp_expert_fwd -> tqp_combine
 *   backward:  tqp_combine_bwd -> tqp_expert_bwd -> tqp_dispatch_bwd [-> tqp_route_bwd]
 *
 * Notation: T tokens, d = d_model, F = per-expert d_ff, E experts, k = top-k, r = adapter rank,
 * N = T*k routed rows, a = t*k + j the flat assignment index of token t's j-th choice,
 * p the row position after the stable sort by expert (perm[p] = a, inv_perm[a] = p).
 *
 * Conventions for EVERY entry point below unless a comment says otherwise:
 *  - All tensor pointers are DEVICE pointers, row-major, contiguous, 16-byte aligned, caller-owned; the
 *    library never frees them and never dereferences them after the call has been enqueued, except the
 *    tqp_weights pointers and the bound workspace, which must stay valid while the ctx uses them, and the
 *    buffers of a tqp_step_host_async step until tqp_step_host_wait has returned for it.
 *  - "bf16" / "fp16" tensors are passed as const void* (2 bytes per element).
 *  - `stream` is a cudaStream_t passed as void*.  Every call only enqueues work on it: no host
 *    synchronisation, no device->host copy.  Expert counts/offsets are consumed on the device.
 *  - Return value: TQP_OK or an error code; nothing throws or aborts.  Host-side argument validation runs
 *    first; CUDA errors map to TQP_ERR_CUDA with the text kept in tqp_last_error(ctx).
 *  - There is NO CPU fallback: without an sm_100 device the calls return TQP_ERR_ARCH / TQP_ERR_CUDA.
 *  - Non-finite inputs: undefined results.
 */
#ifndef TQP_H_
#define TQP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tqp_ctx tqp_ctx; /* opaque; owns only host-side state (descriptors, pointers) */

typedef enum {
    TQP_OK = 0,
    TQP_ERR_ARG = 1,       /* NULL pointer or value out of range */
    TQP_ERR_SHAPE = 2,     /* unsupported shape (see tqp_layer_desc) */
    TQP_ERR_ALIGN = 3,     /* pointer not 16-byte aligned */
    TQP_ERR_WORKSPACE = 4, /* workspace missing or too small */
    TQP_ERR_STATE = 5,     /* call order violated (e.g. expert_bwd without a training-mode expert_fwd) */
    TQP_ERR_ARCH = 6,      /* device is not sm_100 */
    TQP_ERR_CUDA = 7       /* a CUDA runtime/driver call failed; see tqp_last_error */
} tqp_status;

/* Shape of one layer.  Constraints: d % 128 == 0, F % 128 == 0, 1 <= k <= min(E, 32), E <= 1024,
 * r in {8, 16, 32}, vec == 8, codes == 256, T_max * k < 2^31 / 64. */
typedef struct {
    int32_t T_max;    /* largest T any call will pass */
    int32_t d, F, E, k, r;
    int32_t vec;      /* vector length of the quantiser: 8 (BASELINE.json configs[0]) */
    int32_t codes;    /* codebook entries: 256 */
    float lora_scale; /* s in W_eff = deq(W) + s*A*B  (R7; 1.0 in all configs) */
    int32_t training; /* 1: expert_fwd saves G, U, H in the workspace for expert_bwd */
} tqp_layer_desc;

/* Frozen quantised base + trained adapters of all E experts.  All DEVICE pointers.
 * W_eff[in][out] = scale[out] * codebook[idx[out][in/8]][in%8] + lora_scale * (A . B)[in][out]. */
typedef struct {
    const uint8_t *idx_gate, *idx_up; /* [E][F][d/8]  row = output channel, codes along the input dim */
    const uint8_t *idx_down;          /* [E][d][F/8] */
    const void *scale_gate, *scale_up; /* fp16 [E][F] */
    const void *scale_down;            /* fp16 [E][d] */
    const void *codebook;              /* fp16 [256][8], shared by all experts and the three packs */
    const void *A_gate, *A_up;         /* bf16 [E][d][r] */
    const void *B_gate, *B_up;         /* bf16 [E][r][F] */
    const void *A_down;                /* bf16 [E][F][r] */
    const void *B_down;                /* bf16 [E][r][d] */
} tqp_weights;

/* --- lifetime ----------------------------------------------------------------------------------------- */
tqp_status tqp_create(tqp_ctx **out, const tqp_layer_desc *desc); /* validates desc and the device */
void tqp_destroy(tqp_ctx *ctx);
/* Bytes of device scratch the ctx needs (saved G/U/H, permuted rows, adapter projections, tile lists). */
size_t tqp_workspace_bytes(const tqp_layer_desc *desc);
/* Caller allocates (e.g. torch.empty) and lends the workspace; it is zero-filled on `stream`. */
tqp_status tqp_bind_workspace(tqp_ctx *ctx, void *dev_ptr, size_t bytes, void *stream);
/* Records the weight pointers, builds the TMA descriptors over the code indices and converts the codebook
 * to the bf16 lookup table the GEMM mainloop gathers from.  One-time, untimed; needs a bound workspace. */
tqp_status tqp_bind_weights(tqp_ctx *ctx, const tqp_weights *w, void *stream);
/* Options.
 * "gemm_impl": 0 = tcgen05 grouped GEMM on CTA pairs with the dequantised weight operand in tensor memory (default),
 *   1 = CUDA-core scaffold (test reference), 2 = tcgen05 grouped GEMM, one CTA per tile, weight operand through shared
 *   memory (fallback for M % 256 != 0), 3 = CTA pairs, weight operand through shared memory (fallback for K % 128 != 0).
 * "route_impl": 0..3, see tqp_route_info.
 * "fuse_dgu": 1 (default) lets tqp_expert_bwd form the gate / up adapter projections and dB_gate / dB_up in one pass over
 *   dG / dU (r in {16, 32}), 0 keeps the separate passes; same results within fp32 summation order.
 * "time_gemm": 0 / 1, see tqp_gemm_time.
 * "host_chunks": 0 (default) lets tqp_step_host_async choose at run time whether X goes up and is routed in one piece or
 *   in four token chunks; 1 / 4 pin the choice (same results).
 * Unknown names return TQP_ERR_ARG.  (Kernel instrumentation -- "trace", "ablate" -- exists only in builds compiled with
 * -DTQP_TRACE and is not part of this interface.) */
tqp_status tqp_set_option(tqp_ctx *ctx, const char *name, int value);

/* --- forward ------------------------------------------------------------------------------------------ */
/* Router (R1-R5).  logits[t][e] = fmaf-chain over i ascending of
 * float(X[t][i]) * W_r[i][e], then + logit_bias[e] if given; top-k by (-logit, id) (ties -> lower id);
 * topk_w = softmax over the k selected logits.  X bf16 [T][d]; W_r fp32 [d][E]; logit_bias fp32 [E] or
 * NULL; topk_idx int32 [T][k]; topk_w fp32 [T][k]; logits_out fp32 [T][E] or NULL. */
tqp_status tqp_route(tqp_ctx *ctx, int T, const void *X, const float *W_r, const float *logit_bias,
                     int32_t *topk_idx, float *topk_w, float *logits_out, void *stream);
/* How the last tqp_route of this ctx ran (synchronises `stream`).  *screened = 1: the screened router (needs
 * logits_out == NULL, d % 128 == 0, E <= 1024, k <= 32 and X 16-byte aligned; option "route_impl" 0, the default, takes it
 * where it is the faster one -- E > 6 (k + 4) and T E d >= 3e9 --, 2 wherever it can run):
 * approximate logits on the tensor cores with a proven error bound, the canonical fmaf chain only for the experts within
 * that bound of a token's k-th largest, top-k and softmax on those exact values -- topk_idx and topk_w are bit-identical
 * to the dense chain (R1, section 6).  *fallback = 1: the screen's self-check tripped (or a token had more than
 * 64 candidates, e.g. an all-zero row) and the dense chain recomputed the call behind it; the results are the same.
 * "route_impl" 1 = always the dense chain; 3 = as 2 with the self-check forced to fail (exercises the fallback). */
tqp_status tqp_route_info(tqp_ctx *ctx, int *screened, int *fallback, void *stream);
/* Stable counting sort of a = t*k+j by expert id ("expert dispatch").  counts int32 [E];
 * offsets int32 [E+1] (exclusive scan, offsets[E] = N); perm int32 [N]; inv_perm int32 [N].  Also builds
 * the grouped-GEMM tile list inside the workspace. */
tqp_status tqp_dispatch(tqp_ctx *ctx, int T, const int32_t *topk_idx, int32_t *counts, int32_t *offsets,
                        int32_t *perm, int32_t *inv_perm, void *stream);
/* Routed experts: for row p of expert e, x = X[perm[p]/k]:
 * g = x.Wg_eff, u = x.Wu_eff, h = silu(g)*u, Ye[p] = h.Wd_eff.  Ye bf16 [N][d].  Must follow tqp_dispatch
 * with the same T on the same stream (uses its tile list). */
tqp_status tqp_expert_fwd(tqp_ctx *ctx, int T, const void *X, const int32_t *offsets, const int32_t *perm,
                          void *Ye, void *stream);
/* Weighted combine: Y[t] = sum_j topk_w[t][j] * Ye[inv_perm[t*k+j]] (fp32 accumulate, j ascending).
 * Y bf16 [T][d]. */
tqp_status tqp_combine(tqp_ctx *ctx, int T, const void *Ye, const int32_t *inv_perm, const float *topk_w,
                       void *Y, void *stream);

/* --- backward (loss L = sum(Y * dY)) -------------------------------------------------------------------- */
/* dYe[p] = topk_w[a] * dY[t] (bf16 [N][d]);  dtopk_w[a] = <dY[t], Ye[p]> (fp32 [T][k], NULL to skip).
 * perm (int32 [N], the array tqp_dispatch wrote together with inv_perm; NULL allowed): when given, and the ctx is a
 * training ctx with bound weights and r in {16, 32}, dYe is produced by sorted position with a TMA row gather and the
 * adapter projection s * dYe . B_down^T that tqp_expert_bwd needs is computed from the same rows into the workspace
 * (one pass instead of two).  With perm == NULL a plain kernel walks inv_perm; the results are the same. */
tqp_status tqp_combine_bwd(tqp_ctx *ctx, int T, const void *dY, const void *Ye, const int32_t *inv_perm,
                           const int32_t *perm, const float *topk_w, void *dYe, float *dtopk_w, void *stream);
/* Activation gradient through the frozen dequantised weights and weight gradients of the adapters only
 * (PAPER.md L938).  Needs training=1 and the preceding tqp_expert_fwd of the same T.  dXp bf16 [N][d];
 * dA_gate/dA_up fp32 [E][d][r]; dB_gate/dB_up fp32 [E][r][F]; dA_down fp32 [E][F][r]; dB_down fp32
 * [E][r][d]; gradients are overwritten (exactly 0 for experts with no rows).
 * flags: 0, or TQP_BWD_DYE_UNMODIFIED = the caller vouches that dYe is exactly the tensor the directly preceding
 * tqp_combine_bwd (called with perm) on this ctx wrote, unmodified since: its adapter projection is then reused instead of
 * being recomputed from dYe.  TQP_ERR_STATE if no such call preceded or dYe is another pointer.  With flags = 0 nothing
 * from an earlier call is trusted (a caller that adds, say, a shared-expert gradient to dYe in place passes 0). */
#define TQP_BWD_DYE_UNMODIFIED 1
tqp_status tqp_expert_bwd(tqp_ctx *ctx, int T, const void *X, const void *dYe, const int32_t *offsets,
                          const int32_t *perm, void *dXp, float *dA_gate, float *dB_gate, float *dA_up,
                          float *dB_up, float *dA_down, float *dB_down, int flags, void *stream);
/* dX[t] = sum_j dXp[inv_perm[t*k+j]] (fp32 accumulate, j ascending); dX bf16 [T][d]. */
tqp_status tqp_dispatch_bwd(tqp_ctx *ctx, int T, const void *dXp, const int32_t *inv_perm, void *dX,
                            void *stream);
/* Router gradient with the selection held constant: dl_j = w_j (dw_j - sum_i w_i dw_i);
 * dX[t] += sum_j dl_j W_r[:,e_j] (dX bf16 [T][d], read-modify-write); dW_r[:,e] = sum X[t] dl (fp32 [d][E],
 * overwritten).  Uses the perm/offsets of the preceding tqp_dispatch for a deterministic reduction. */
tqp_status tqp_route_bwd(tqp_ctx *ctx, int T, const void *X, const float *W_r, const int32_t *topk_idx,
                         const float *topk_w, const float *dtopk_w, const int32_t *offsets,
                         const int32_t *perm, void *dX, float *dW_r, void *stream);

/* --- whole step through HOST buffers (end-to-end measurement) ------------------------------------------- */
/* Copies X and dY (bf16 [T][d], pinned HOST memory) to the device, runs the whole forward+backward chain
 * above on `stream` and copies Y and dX (bf16 [T][d]) back to the HOST buffers.  W_r / logit_bias and the
 * adapter-gradient outputs are DEVICE pointers as above (dW_r may be NULL to skip tqp_route_bwd).
 * Synchronises `stream` before returning.  The device-side staging of these calls (two upload sets, the routing arrays,
 * Ye / dYe / dXp: 1.7 GB at configs[2]) is NOT part of the caller's workspace: the library allocates it on the first call
 * and frees it in tqp_destroy, so a caller of the stepwise API never pays for it. */
tqp_status tqp_step_host(tqp_ctx *ctx, int T, const void *X_host, const void *dY_host, const float *W_r,
                         const float *logit_bias, void *Y_host, void *dX_host, float *dA_gate,
                         float *dB_gate, float *dA_up, float *dB_up, float *dA_down, float *dB_down,
                         float *dW_r, void *stream);

/* The same step without the final synchronisation: everything is enqueued (kernels on `stream`, copies on the ctx's
 * two copy streams) and the call returns.  A second call may follow at once: its uploads use the other of two device
 * staging sets and travel while the first step's kernels run, its kernels follow on `stream`, and the first step's dX
 * download overlaps its forward pass - the pipelining a data loader gives a training loop.  The host buffers of a step
 * belong to the library until tqp_step_host_wait has returned for it: at most two steps may be in flight.
 * tqp_step_host_wait(ctx, age) blocks the host until the latest (age 0) or the previous (age 1) enqueued step has
 * delivered Y_host / dX_host and finished its kernels (gradients included); returns at once if there is no such step.
 * Errors as tqp_step_host; TQP_ERR_ARG for another age. */
tqp_status tqp_step_host_async(tqp_ctx *ctx, int T, const void *X_host, const void *dY_host, const float *W_r,
                               const float *logit_bias, void *Y_host, void *dX_host, float *dA_gate,
                               float *dB_gate, float *dA_up, float *dB_up, float *dA_down, float *dB_down,
                               float *dW_r, void *stream);
tqp_status tqp_step_host_wait(tqp_ctx *ctx, int age);

/* --- paper-faithful router variant and loss-free balance controller -------------- */
/* PAPER.md L224 (§3.4): "Routing scores are produced by a sigmoid, expert selection is biased by a per-expert routing
 * logit bias".  logits as in tqp_route (canonical fmaf chain, NO bias added); selection = the k largest keys
 * logits[t][e] + select_bias[e] (fp32 add; ties -> lower id; select_bias fp32 [E] or NULL); topk_s[t][j] =
 * sigmoid(logit) of the UNBIASED selected logit; topk_w = topk_s / sum_j topk_s (summed in ascending j) -- DESIGN.md
 * R21, R22.  topk_idx int32 [T][k]; topk_w, topk_s fp32 [T][k]; logits_out fp32 [T][E] or NULL.  All DEVICE pointers.
 * With logits_out == NULL the screened router runs under the same rule as in tqp_route (tqp_route_info reports it). */
tqp_status tqp_route_sigmoid(tqp_ctx *ctx, int T, const void *X, const float *W_r, const float *select_bias,
                             int32_t *topk_idx, float *topk_w, float *topk_s, float *logits_out, void *stream);
/* Router backward for tqp_route_sigmoid (selection held constant, the bias has no gradient):
 * dl_j = (dtopk_w_j - sum_i topk_w_i dtopk_w_i) * topk_w_j * (1 - topk_s_j), then as tqp_route_bwd:
 * dX[t] += sum_j dl_j W_r[:,e_j] (dX bf16 [T][d], accumulated in place), dW_r[:,e] = sum_{rows of e} X[t] dl
 * (fp32 [d][E], overwritten). */
tqp_status tqp_route_sigmoid_bwd(tqp_ctx *ctx, int T, const void *X, const float *W_r, const int32_t *topk_idx,
                                 const float *topk_w, const float *topk_s, const float *dtopk_w, const int32_t *offsets,
                                 const int32_t *perm, void *dX, float *dW_r, void *stream);
/* One step of the loss-free bias controller over the dispatch counts of a batch (§10.5, L1097 Table 29,
 * L1516 Table 37): load_e = counts[e] / sum(counts), tau = 1/E.
 * mode 0 (sign-based, 5B/9B):  bias[e] += gamma * sign(tau - load_e).
 * mode 1 (three-tier band with quadratic boost, 120B; R23): inside [cap_lo, cap_hi] as mode 0; load > cap_hi:
 *   bias[e] -= gamma * (1 + ((load - cap_hi)/tau)^2); load < cap_lo: bias[e] += gamma * (1 + ((cap_lo - load)/tau)^2);
 *   cap_lo <= 0 selects tau^2 / cap_hi.  counts int32 [E] (device, e.g. from tqp_dispatch); bias fp32 [E], in place. */
tqp_status tqp_bias_update(tqp_ctx *ctx, const int32_t *counts, float *bias, int mode, float gamma, float cap_hi,
                           float cap_lo, void *stream);

/* --- consolidation ---------------------------------------------------------- */
/* PAPER.md L1110 (10.6) "The trained adapter is merged into the base weights, the result is materialized as bf16";
 * L1481.  Writes the merged, ordinary bf16 weights of experts e0 .. e0 + n_experts - 1 of one pack
 * (0 = gate, 1 = up, 2 = down):
 *   W_out[e - e0][out][in] = bf16( scale[out] * codebook[idx[out][in/8]][in%8] + lora_scale * sum_q A[in][q] B[q][out] )
 * computed in fp32 with one rounding; row = output channel, so that y = x . W^T is the dense layer (gate / up:
 * out = F, in = d; down: out = d, in = F).  W_out: DEVICE bf16 [n_experts][out][in], caller-owned (5.2 MB per expert
 * and pack at d = 2560, F = 1024: consolidate in expert ranges).  Needs bound weights; reads them, writes nothing else.
 * Errors: TQP_ERR_STATE without weights, TQP_ERR_ARG for a bad pack / range / NULL. */
tqp_status tqp_consolidate(tqp_ctx *ctx, int pack, int e0, int n_experts, void *W_out, void *stream);

/* --- TurboQuant-MSE base --------------------------------------------------- */
/* PAPER.md L944-946 (9.2): "the quantizer separates scale from direction, normalizes the vector and stores its norm,
 * applies a seeded random orthogonal rotation, and then quantizes each rotated coordinate independently against a scalar
 * codebook ... The rotation is a signed Hadamard transform when the dimension is a power of two and a QR rotation from a
 * Gaussian matrix with sign fixing otherwise.  Reconstruction looks up the codebook values and rescales by the stored
 * norm."  L946: 8-bit, "the per-expert weight packs quantized row by row" (row = output channel, width n = the pack's
 * input width).  Storage: one uint8 code per rotated coordinate, one fp32 norm per row (the paper prints no dtype for
 * the norm: DESIGN.md R24).
 *
 * One rotated space: y = R u.  hadamard = 1: R = H_n diag(signs) / sqrt(n), H_n the Sylvester matrix, n a power of two;
 * hadamard = 0: R a dense orthogonal matrix (e.g. from tqp_tq_rotation_qr).  n % 64 == 0, 64 <= n <= 8192 (dense rotations of
 * activations additionally n % 128 == 0).  The seeded random draws (signs, Gaussian matrix) are the caller's inputs.
 * All pointers DEVICE; they must stay valid while any call or bound layer uses the space.  For a dense R the library
 * keeps derived device copies (bf16 R, R^T; fp64 R^T) inside the ctx, keyed by the R pointer, until tqp_destroy. */
typedef struct {
    int32_t n;
    int32_t hadamard;
    const int8_t *signs;  /* int8 [n], +1 / -1 (hadamard = 1), else NULL */
    const double *R;      /* fp64 [n][n] row-major (hadamard = 0), else NULL */
    const double *levels; /* fp64 [256], ascending: the Lloyd-Max levels of the coordinate law in dimension n */
} tqp_tq_space;
/* HOST: the 2^bits Lloyd-Max levels of f_n(y) ~ (1 - y^2)^((n-3)/2) on [-1, 1] (L944: "computed analytically from that law"),
 * ascending, into the HOST array levels[2^bits].  n >= 8, 1 <= bits <= 8. */
tqp_status tqp_tq_levels(int n, int bits, double *levels);
/* HOST: the sign-fixed Q of the QR factorisation of G (HOST fp64 [n][n] row-major, the caller's seeded Gaussian draw):
 * the unique orthogonal Q with G = Q Rr, diag(Rr) > 0, into the HOST array R_out[n][n] (L946 "QR rotation ... with sign fixing"). */
tqp_status tqp_tq_rotation_qr(int n, const double *G, double *R_out);
/* Rotation of activations: Y[row] = R X[row] (inverse = 0) or R^T X[row] (inverse = 1); X, Y bf16 [rows][n], Y may be X only for
 * hadamard spaces.  Hadamard: one FWHT pass (HBM-bound); dense: a bf16 tensor-core product with fp32 accumulation. */
tqp_status tqp_rotate(tqp_ctx *ctx, const tqp_tq_space *space, const void *X, long long rows, void *Y, int inverse, void *stream);
/* Encoder, row by row (L944-946): norms[row] = |W[row]|, codes[row][j] = index of the Lloyd-Max cell of (R W[row] / norm)_j
 * (a coordinate on a cell boundary takes the lower code; a zero row: norm 0 and the codes of y = 0).  W fp32 [rows][n];
 * codes uint8 [rows][n]; norms fp32 [rows].  Norm, rotation and cell search run in fp64. */
tqp_status tqp_tq_encode(tqp_ctx *ctx, const tqp_tq_space *space, const float *W, long long rows, uint8_t *codes, float *norms,
                         void *stream);
/* Reconstruction (L946): W[row] = norms[row] * (levels[codes[row]] R), fp32 [rows][n]. */
tqp_status tqp_tq_decode(tqp_ctx *ctx, const tqp_tq_space *space, const uint8_t *codes, const float *norms, long long rows, float *W,
                         void *stream);
/* Flush (PAPER.md L966 9.4: "periodically fold the adapter delta into the base, reset the adapter factors"; L1047-1061 10.3,
 * Table 28: "the mean adapter norm ... and the share of each effective weight still coming from the frozen base") of one
 * pack of n_experts experts, in place:
 *   W = decode(codes, norms);  W_merged = W + lora_scale (A B)^T;  (codes, norms) <- encode(W_merged);  B <- 0;
 *   A <- A_new if A_new != NULL.
 * The fold and the re-quantisation run in the ROTATED space (R W_merged = norm levels[codes] + lora_scale (R A) B column
 * by column), in fp64, without materialising a weight in HBM.  codes uint8 [n_experts][out_dim][n]; norms fp32
 * [n_experts][out_dim]; A bf16 [n_experts][n][r]; B bf16 [n_experts][r][out_dim]; A_new like A or NULL; telemetry fp32
 * [n_experts][2] or NULL: (|lora_scale A B|_F, |W|_F / (|W|_F + |lora_scale A B|_F)) of the state BEFORE the fold
 * (R26).  1 <= r <= 32. */
tqp_status tqp_tq_flush(tqp_ctx *ctx, const tqp_tq_space *space, int n_experts, int out_dim, int r, float lora_scale, uint8_t *codes,
                        float *norms, void *A, void *B, const void *A_new, float *telemetry, void *stream);

/* The routed-expert layer over a TurboQuant base.  Frozen base: one code per rotated coordinate and one norm per row;
 * W_eff[in][out] = norm[out] * (levels[codes[out]] R)[in] + lora_scale * (A . B)[in][out]  with R, levels of the pack's
 * input space (space_d for gate / up, space_F for down).  Adapters as in tqp_weights (unrotated).  All DEVICE pointers. */
typedef struct {
    const uint8_t *codes_gate, *codes_up; /* [E][F][d] */
    const uint8_t *codes_down;            /* [E][d][F] */
    const float *norm_gate, *norm_up;     /* fp32 [E][F] */
    const float *norm_down;               /* fp32 [E][d] */
    tqp_tq_space space_d, space_F;
    const void *A_gate, *A_up;            /* bf16 [E][d][r] */
    const void *B_gate, *B_up;            /* bf16 [E][r][F] */
    const void *A_down;                   /* bf16 [E][F][r] */
    const void *B_down;                   /* bf16 [E][r][d] */
} tqp_tq_weights;
/* Binds a TurboQuant base in place of tqp_bind_weights; afterwards tqp_expert_fwd / tqp_expert_bwd / tqp_dispatch_bwd (and the
 * tqp_step_host calls) run the same layer over it.  How: the rotation is applied ONCE to the activations (x' = R_d x on the
 * T token rows before the gather; h' = R_F h after the SwiGLU), the grouped GEMM's mainloop then looks each code up in a
 * 256-entry scalar table and scales by the row norm -- no weight is materialised -- and the adapters' input side is
 * carried into the rotated space (A' = R A, so that x . A = x' . A'); gradients come back through R^T.  Two things differ
 * for the caller: (1) with a TurboQuant base bound, the dXp tensor tqp_expert_bwd returns holds the gradient in the
 * ROTATED input space, and tqp_dispatch_bwd undoes the rotation after the token sum (the rotation is linear);
 * (2) needs r in {16, 32}, d % 256 == 0, F % 256 == 0, training ctx or not.  The library allocates its own device
 * buffers for the rotated activations / adapters (freed by tqp_destroy or the next bind).  TQP_ERR_SHAPE for unsupported
 * shapes or spaces whose n is not d / F. */
tqp_status tqp_bind_weights_tq(tqp_ctx *ctx, const tqp_tq_weights *w, void *stream);

/* --- introspection ------------------------------------------------------------------------------------- */
/* Device pointers of workspace tensors, for tests: "G","U","H" bf16 [N][F]; "Xp" bf16 [N][d];
 * "dH","dG","dU" bf16 [N][F]; "num_tiles" int32 [1].  NULL if unknown. */
void *tqp_debug_buffer(tqp_ctx *ctx, const char *name);
/* --- dispatch without any allocation ------------------------------------------------------------------------ */
/* tqp_dispatch ("expert dispatch": stable counting sort of a = t*k+j by expert id) for callers that cannot
 * allocate -- code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No ctx, no workspace:
 * the call allocates nothing on the host or the device and calls no allocating routine.  Its scratch (per-chunk
 * histograms) is a fixed 4 MiB __device__ array inside the library, which every GPU that loads the library holds until
 * the process exits.  topk_idx int32 [T][k] (values in [0, E)); counts int32 [E]; offsets int32 [E+1]; perm, inv_perm
 * int32 [T*k]: all DEVICE pointers of the current device, caller-owned; results equal tqp_dispatch's bit for bit (the
 * grouped-GEMM tile list is not built).  Limits: 1 <= E <= 1024, 1 <= k <= min(32, E), T*k < 2^25 (TQP_ERR_ARG) and
 * ceil(T*k / 256) * E <= tqp_dispatch_noalloc_capacity() = 1 048 576 (TQP_ERR_SHAPE; e.g. T = 16384, k = 12, E = 460
 * uses a third of it).  All calls on a device share the array: calls on one stream are ordered and safe, calls that
 * OVERLAP on the GPU (other streams, a graph replayed beside a live call) race and give garbage.  Nothing in it has to be
 * cleared: every entry a call reads it has written before.  The first call on a device also looks the array's device address
 * up (cudaGetSymbolAddress, once per device): make that call before a stream capture begins.  Errors: the codes above,
 * TQP_ERR_CUDA for a failed look-up or launch;
 * text in tqp_dispatch_noalloc_error() (per thread). */
tqp_status tqp_dispatch_noalloc(int T, int k, int E, const int32_t *topk_idx, int32_t *counts, int32_t *offsets,
                                int32_t *perm, int32_t *inv_perm, void *stream);
size_t tqp_dispatch_noalloc_capacity(void);
const char *tqp_dispatch_noalloc_error(void);

/* Measurement hook (the >= 50 % target applies to the grouped-GEMM kernels' own time).  After
 * tqp_set_option(ctx, "time_gemm", 1) every grouped-GEMM launch is bracketed by CUDA events on its stream.
 * tqp_gemm_time waits for the recorded events, returns the summed device time in milliseconds and the number of
 * GEMM launches since the previous call, and resets the record (at most 4096 launches are kept). */
tqp_status tqp_gemm_time(tqp_ctx *ctx, float *ms_total, int *launches);
/* Same record, per launch: writes up to `cap` per-launch times (ms, launch order) into the HOST array ms_each
 * and the launch count into *launches; resets the record. */
tqp_status tqp_gemm_times(tqp_ctx *ctx, float *ms_each, int cap, int *launches);
/* Kernels launched by the last call on this ctx (for bench.py's gpu_launches). */
int tqp_last_launch_count(const tqp_ctx *ctx);
const char *tqp_status_string(tqp_status s);
const char *tqp_last_error(const tqp_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* TQP_H_ */
