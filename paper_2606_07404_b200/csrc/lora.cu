// Adapter side products of the TQP layer (rank-r adapter on each weight pack, only the adapters train).
//   rows_proj : P_w[p][0..r) = s * row(p) . W_w[e]      (x.A_g | x.A_u, h.A_d forward;  dy.B^T backward)  -> [N][64] bf16
//               row(p) is either in[p] or a GATHERED (and optionally gate-weighted) row in[perm[p]/k] * w[perm[p]],
//               which the kernel also writes through to the dense permuted tensor (Xp = gather(X), dYe = w . gather(dY)):
//               the token permutation, the combine backward (a7) and the adapter projections that
//               follow them read their rows from HBM once instead of two or three times.
//   rows_wgrad: grad_w[e] = sum_{p in e} small_w[p]^T big[p]   (dA = x^T z, dB = (xA)^T dy), fp32, deterministic
// Both are tall-skinny grouped contractions whose cost is streaming the [N][K] operand once: bound = HBM.  Rows stream
// through a cp.async ring; the contraction itself is warp-level bf16 MMA (ldmatrix + mma.sync m16n8k16, fp32
// accumulate) -- the legacy HMMA path is enough here because the kernels need < 10 % of its rate at HBM speed.
#include "common.cuh"
#include "tc_ptx.cuh"

namespace tqp {

__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// four 8x8 b16 matrices; lane l supplies the row address of matrix l/8, row l%8 (shared-space address)
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t (&r)[4]) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
// D[16x8] += A[16x16] B[16x8]; bf16 operands, fp32 accumulate
__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// ---- projections ------------------------------------------------------------------------------------------------
// Rows go global -> registers (LDG.128, two K-chunks ahead) -> shared (+ straight from the registers to the dense
// permuted tensor in the gathered variants).  cp.async was tried first for the rows: its 16-byte requests cost two
// 32-byte L2 sectors each (ncu: lts read sectors = 1.9 x the bytes asked for) and made the kernel L2-throughput-bound;
// 256-byte cp.async.bulk row copies were slower still.  Warp-wide LDG.128 moves exactly the sectors it needs.  The
// small adapter chunks (shared by the 128 rows of the CTA) keep the cp.async ring: they cost no registers.
constexpr int PJ_ROWS = 128;         // rows per CTA (8 warps x 16)
constexpr int PJ_THREADS = 256;
constexpr int PJ_KC = 64;            // K-chunk per step (128 contiguous bytes of every row)
constexpr int PJ_LD = PJ_KC + 8;     // padded smem row (bf16): conflict-free ldmatrix
constexpr int PJ_CH = PJ_ROWS * PJ_KC / 8 / PJ_THREADS;   // 16-byte row chunks per thread per step
constexpr int PJ_D = 3;              // register sets: chunk kc+2 is in flight while chunk kc is multiplied
constexpr int PJ_WST = 3;            // adapter-chunk ring

struct ProjArgs {
    const bf16 *in;        // source rows [*][K]
    const int32_t *perm;   // != nullptr: row(p) = in[perm[p] / k]   (else in[p])
    const float *roww;     // != nullptr (needs perm): row(p) *= roww[perm[p]], rounded to bf16
    bf16 *through;         // != nullptr: row(p) is also written to through[p][K]
    const bf16 *W[2];      // adapter matrices of all experts
    bf16 *out[2];          // [N][kLoraPad]
    int K, k;
    float s;
    int ablate;            // timing experiments only (tqp_set_option "ablate"): 256 no write-through, 512 no MMA, 1024 no row loads
};

template <int R, int NW, bool KR>
struct ProjCfg {
    static constexpr int RT = R * NW;
    static constexpr int WLD = KR ? RT + 8 : PJ_LD;                  // KR: Ws[KC][RT+8]   else: Ws[RT][KC+8]
    static constexpr int ROWS_BYTES = PJ_ROWS * PJ_LD * 2;
    static constexpr int W_CHUNKS = KR ? PJ_KC * RT / 8 : RT * PJ_KC / 8;   // 16-byte pieces of the adapter chunk
    static constexpr int W_BYTES = ((KR ? PJ_KC * WLD : RT * WLD) * 2 + 127) / 128 * 128;
    static constexpr int OFF_W = 2 * ROWS_BYTES;
    static constexpr int SMEM = OFF_W + PJ_WST * W_BYTES;
};

// L2 eviction priorities: gathered source rows (X, dY: 42 MB, each row reused k times) should stay resident while
// the 0.5 GB of read-once / write-once permuted rows stream through.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint4 ldg128_hint(const void *p, uint64_t pol) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ void stg128_hint(void *p, const uint4 &v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v4.u32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(pol)
                 : "memory");
}

// grid = (max_tiles, kTileRows / 128), block = 256.  KR: W_e is [K][R] (x.A), else [R][K] (dy.B^T).
template <int R, int NW, bool KR>
__global__ void __launch_bounds__(PJ_THREADS, 2) rows_proj_kernel(const __grid_constant__ ProjArgs a, const Tile *__restrict__ tiles,
                                                                  const int32_t *__restrict__ num_tiles) {
    using C = ProjCfg<R, NW, KR>;
    extern __shared__ __align__(128) uint8_t pj_smem[];   // used directly: a pointer rebuilt from an integer would
                                                          // lose its address space (generic LD.E instead of LDS/ldmatrix)
    if ((int)blockIdx.x >= *num_tiles) return;
    const Tile t = tiles[blockIdx.x];
    const int rbase = blockIdx.y * PJ_ROWS;
    const int valid = min(PJ_ROWS, t.rows - rbase);
    if (valid <= 0) return;
    const int row0 = t.row0 + rbase;
    const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(pj_smem);
    const int K = a.K;

    // this thread's row chunks: rows rr + RSTEP i (i < PJ_CH), 16-byte chunk rc of every K-chunk
    constexpr int TPR = PJ_KC / 8, RSTEP = PJ_THREADS / TPR;
    const int rr = tid / TPR, rc = tid % TPR;
    const bf16 *src[PJ_CH];
    float roww[PJ_CH];
#pragma unroll
    for (int i = 0; i < PJ_CH; ++i) {
        const int r = rr + RSTEP * i;
        src[i] = nullptr;   // rows past `valid` are not loaded (zeros; their outputs are never stored)
        roww[i] = 1.f;
        if (r < valid && !TQP_DBG(a.ablate & 1024)) {
            int srow = row0 + r;
            if (a.perm) {
                const int as = a.perm[srow];
                srow = as / a.k;
                if (a.roww) roww[i] = a.roww[as];
            }
            src[i] = a.in + (size_t)srow * K + rc * 8;
        }
    }
    auto issue_w = [&](int kc) {   // adapter chunk kc -> ring slot kc % PJ_WST
        const uint32_t w_s = sbase + C::OFF_W + (kc % PJ_WST) * C::W_BYTES;
        for (int v = tid; v < C::W_CHUNKS; v += PJ_THREADS) {
            if (KR) {   // W_w[e][k][R]: piece = (k, w, 8 columns)
                const int kk = v / (C::RT / 8), cc = v % (C::RT / 8), w = (cc * 8) / R, q0 = (cc * 8) % R;
                cp_async16(w_s + (kk * C::WLD + cc * 8) * 2, a.W[w] + ((size_t)t.expert * K + kc * PJ_KC + kk) * R + q0, 16);
            } else {    // W_w[e][q][K]: piece = (w, q, 8 k)
                const int n = v / (PJ_KC / 8), cc = v % (PJ_KC / 8), w = n / R, q = n % R;
                cp_async16(w_s + (n * C::WLD + cc * 8) * 2, a.W[w] + ((size_t)t.expert * R + q) * K + kc * PJ_KC + cc * 8, 16);
            }
        }
    };

    const uint64_t pol_ld = a.perm ? l2_policy_evict_last() : l2_policy_evict_first(), pol_st = l2_policy_evict_first();
    uint4 pre[PJ_D][PJ_CH];
    auto fetch = [&](int kc, uint4 (&rows)[PJ_CH]) {
#pragma unroll
        for (int i = 0; i < PJ_CH; ++i) rows[i] = src[i] ? ldg128_hint(src[i] + (size_t)kc * PJ_KC, pol_ld) : make_uint4(0, 0, 0, 0);
    };

    float acc[C::RT / 8][4];
#pragma unroll
    for (int n = 0; n < C::RT / 8; ++n)
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[n][q] = 0.f;

    const int nk = K / PJ_KC;
    const bool rewrite = a.roww != nullptr, thru = a.through != nullptr && !TQP_DBG(a.ablate & 256);
#pragma unroll
    for (int s = 0; s < PJ_D - 1; ++s) {
        if (s < nk) { fetch(s, pre[s]); issue_w(s); }
        cp_async_commit();
    }

    auto step = [&](int kc, uint4 (&rows)[PJ_CH], uint4 (&rows_nx)[PJ_CH]) {
        if (kc + PJ_D - 1 < nk) fetch(kc + PJ_D - 1, rows_nx);
        const uint32_t rows_s = sbase + (kc & 1) * C::ROWS_BYTES;
#pragma unroll
        for (int i = 0; i < PJ_CH; ++i) {
            const int r = rr + RSTEP * i;
            uint4 v = rows[i];
            if (rewrite) {   // gate weight, rounded to bf16 (the value the dH GEMM reads back from dYe)
                uint32_t *vp = reinterpret_cast<uint32_t *>(&v);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    float2 f = bf16x2_to_float2(vp[q]);
                    vp[q] = float2_to_bf16x2(roww[i] * f.x, roww[i] * f.y);
                }
            }
            ptx::sts128(rows_s + (r * PJ_LD + rc * 8) * 2, v);
            if (thru && r < valid) stg128_hint(a.through + (size_t)(row0 + r) * K + kc * PJ_KC + rc * 8, v, pol_st);
        }
        cp_async_wait<PJ_WST - 2>();   // adapter chunk kc has landed (chunk kc + 1 may still be in flight)
        __syncthreads();               // rows + adapter chunk kc visible; everyone is past the MMAs of step kc - 1
        if (kc + PJ_WST - 1 < nk) issue_w(kc + PJ_WST - 1);
        cp_async_commit();
        if (warp * 16 < valid && !TQP_DBG(a.ablate & 512)) {
            const uint32_t w_s = sbase + C::OFF_W + (kc % PJ_WST) * C::W_BYTES;
            const uint32_t a_addr = rows_s + ((warp * 16 + lane % 16) * PJ_LD + (lane / 16) * 8) * 2;
            const uint32_t b_addr = KR ? w_s + ((lane % 8 + ((lane / 8) % 2) * 8) * C::WLD + (lane / 16) * 8) * 2
                                       : w_s + (((lane / 16) * 8 + lane % 8) * C::WLD + ((lane / 8) % 2) * 8) * 2;
#pragma unroll
            for (int kk = 0; kk < PJ_KC; kk += 16) {
                uint32_t af[4];
                ldsm_x4(a_addr + kk * 2, af);
#pragma unroll
                for (int np = 0; np < C::RT / 16; ++np) {
                    uint32_t bq[4];
                    if (KR) ldsm_x4_t(b_addr + (kk * C::WLD + np * 16) * 2, bq);
                    else ldsm_x4(b_addr + (np * 16 * C::WLD + kk) * 2, bq);
                    mma16816(acc[2 * np], af, bq[0], bq[1]);
                    mma16816(acc[2 * np + 1], af, bq[2], bq[3]);
                }
            }
        }
    };
    // Register sets rotate with compile-time indices.  The main loop runs whole triples without conditions so that the
    // three sets keep fixed registers (guarding every step made the compiler merge the sets with moves at the joins).
    int kc = 0;
    for (; kc + PJ_D <= nk; kc += PJ_D) {
        step(kc, pre[0], pre[2]);
        step(kc + 1, pre[1], pre[0]);
        step(kc + 2, pre[2], pre[1]);
    }
    if (kc < nk) {
        step(kc, pre[0], pre[2]);
        if (kc + 1 < nk) step(kc + 1, pre[1], pre[0]);
    }
    cp_async_wait<0>();
    if (warp * 16 < valid) {   // accumulator layout: rows lane/4 (+8), columns 8 n + 2 (lane%4) + {0,1}
#pragma unroll
        for (int n = 0; n < C::RT / 8; ++n) {
            const int col = n * 8 + (lane % 4) * 2, w = col / R, q = col % R;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = warp * 16 + lane / 4 + 8 * h;
                if (r < valid)
                    *reinterpret_cast<uint32_t *>(a.out[w] + (size_t)(row0 + r) * kLoraPad + q) =
                        float2_to_bf16x2(a.s * acc[n][2 * h], a.s * acc[n][2 * h + 1]);
            }
        }
    }
}

template <int R, int NW, bool KR>
static tqp_status launch_proj_t(tqp_ctx *c, const ProjArgs &a, cudaStream_t st) {
    using C = ProjCfg<R, NW, KR>;
    if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&rows_proj_kernel<R, NW, KR>), C::SMEM)) return st_attr;
    dim3 grid(c->max_tiles, kTileRows / PJ_ROWS);
    rows_proj_kernel<R, NW, KR><<<grid, PJ_THREADS, C::SMEM, st>>>(a, c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles));
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// ---- plain projections of a dense workspace tensor, rows by TMA --------------------------------------------------------
// h.A_d, dG.B_g^T, dU.B_u^T: the rows are a dense [N][K] tensor the grouped GEMM already has a tensor map for (box
// 64 columns x 128 rows, 128-byte swizzle).  One thread issues one TMA load per K-chunk into a 5-deep ring (16 KB a stage,
// two CTAs per SM: 128 KB of rows in flight per SM against 64 KB in the register-staged kernel, which these HBM-latency-
// bound passes need); ldmatrix reads the swizzled tile (16-byte chunk c of row r sits at chunk c ^ (r & 7)).
constexpr int PT_NST = 5;
template <int R, bool KR>
struct ProjTmaCfg {
    static constexpr int WLD = KR ? R + 8 : PJ_LD;
    static constexpr int ROWS_BYTES = PJ_ROWS * PJ_KC * 2;                                   // 16 KB, unpadded (swizzled)
    static constexpr int W_CHUNKS = KR ? PJ_KC * R / 8 : R * PJ_KC / 8;
    static constexpr int W_BYTES = ((KR ? PJ_KC * WLD : R * WLD) * 2 + 127) / 128 * 128;
    static constexpr int OFF_W = PT_NST * ROWS_BYTES;
    static constexpr int SMEM = OFF_W + PT_NST * W_BYTES + 1024;
};

struct ProjTmaArgs {
    CUtensorMap map;       // rows [*][K], box {64, 128}, SWIZZLE_128B
    const bf16 *W;         // adapter matrix of all experts
    bf16 *out;             // [N][kLoraPad]
    int K;
    float s;
};

template <int R, bool KR>
__global__ void __launch_bounds__(PJ_THREADS, 2) rows_proj_tma_kernel(const __grid_constant__ ProjTmaArgs a, const Tile *__restrict__ tiles,
                                                                      const int32_t *__restrict__ num_tiles) {
    using C = ProjTmaCfg<R, KR>;
    using namespace ptx;
    extern __shared__ uint8_t pt_smem_raw[];
    __shared__ __align__(8) uint64_t s_full[PT_NST];
    if ((int)blockIdx.x >= *num_tiles) return;
    const Tile t = tiles[blockIdx.x];
    const int rbase = blockIdx.y * PJ_ROWS;
    const int valid = min(PJ_ROWS, t.rows - rbase);
    if (valid <= 0) return;
    const int row0 = t.row0 + rbase;
    const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
    const uint32_t sbase = (smem_u32(pt_smem_raw) + 1023u) & ~1023u;   // shared-space ADDRESS arithmetic only (TMA / ldmatrix / cp.async)
    const uint32_t bar0 = smem_u32(s_full);
    const int K = a.K, nk = K / PJ_KC;
    if (tid == 0) {
        for (int s = 0; s < PT_NST; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_init_fence();
    }
    __syncthreads();
    auto issue = [&](int kc) {   // rows by TMA (one thread), adapter chunk by cp.async (everyone)
        const int st = kc % PT_NST;
        if (tid == 0) {
            mbar_expect_tx(bar0 + 8 * st, C::ROWS_BYTES);
            tma_load_2d(sbase + st * C::ROWS_BYTES, &a.map, kc * PJ_KC, row0, bar0 + 8 * st);
        }
        const uint32_t w_s = sbase + C::OFF_W + st * C::W_BYTES;
        for (int v = tid; v < C::W_CHUNKS; v += PJ_THREADS) {
            if (KR) {   // W[e][k][R]
                const int kk = v / (R / 8), cc = v % (R / 8);
                cp_async16(w_s + (kk * C::WLD + cc * 8) * 2, a.W + ((size_t)t.expert * K + kc * PJ_KC + kk) * R + cc * 8, 16);
            } else {    // W[e][q][K]
                const int q = v / (PJ_KC / 8), cc = v % (PJ_KC / 8);
                cp_async16(w_s + (q * C::WLD + cc * 8) * 2, a.W + ((size_t)t.expert * R + q) * K + kc * PJ_KC + cc * 8, 16);
            }
        }
    };
    float acc[R / 8][4];
#pragma unroll
    for (int n = 0; n < R / 8; ++n)
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[n][q] = 0.f;
    for (int s = 0; s < PT_NST - 1; ++s) {
        if (s < nk) issue(s);
        cp_async_commit();
    }
    const int arow = warp * 16 + lane % 16;   // this lane's row of the A fragment (ldmatrix x4)
    for (int kc = 0; kc < nk; ++kc) {
        const int st = kc % PT_NST;
        mbar_wait(bar0 + 8 * st, (kc / PT_NST) & 1);
        cp_async_wait<PT_NST - 2>();
        __syncthreads();   // chunk kc visible to everyone; everyone is past the MMAs of chunk kc - 1 (its stage is refilled below)
        if (kc + PT_NST - 1 < nk) issue(kc + PT_NST - 1);
        cp_async_commit();
        if (warp * 16 < valid) {
            const uint32_t rows_s = sbase + st * C::ROWS_BYTES, w_s = sbase + C::OFF_W + st * C::W_BYTES;
            const uint32_t b_addr = KR ? w_s + ((lane % 8 + ((lane / 8) % 2) * 8) * C::WLD + (lane / 16) * 8) * 2
                                       : w_s + (((lane / 16) * 8 + lane % 8) * C::WLD + ((lane / 8) % 2) * 8) * 2;
#pragma unroll
            for (int kk = 0; kk < PJ_KC; kk += 16) {
                uint32_t af[4];
                ldsm_x4(rows_s + arow * 128 + ((((kk >> 3) + (lane >> 4)) ^ (arow & 7)) << 4), af);
#pragma unroll
                for (int np = 0; np < R / 16; ++np) {
                    uint32_t bq[4];
                    if (KR) ldsm_x4_t(b_addr + (kk * C::WLD + np * 16) * 2, bq);
                    else ldsm_x4(b_addr + (np * 16 * C::WLD + kk) * 2, bq);
                    mma16816(acc[2 * np], af, bq[0], bq[1]);
                    mma16816(acc[2 * np + 1], af, bq[2], bq[3]);
                }
            }
        }
    }
    cp_async_wait<0>();
    if (warp * 16 < valid) {
#pragma unroll
        for (int n = 0; n < R / 8; ++n) {
            const int q = n * 8 + (lane % 4) * 2;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = warp * 16 + lane / 4 + 8 * h;
                if (r < valid)
                    *reinterpret_cast<uint32_t *>(a.out + (size_t)(row0 + r) * kLoraPad + q) =
                        float2_to_bf16x2(a.s * acc[n][2 * h], a.s * acc[n][2 * h + 1]);
            }
        }
    }
}

template <int R, bool KR>
static tqp_status launch_proj_tma_t(tqp_ctx *c, const ProjTmaArgs &a, cudaStream_t st) {
    using C = ProjTmaCfg<R, KR>;
    if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&rows_proj_tma_kernel<R, KR>), C::SMEM)) return st_attr;
    dim3 grid(c->max_tiles, kTileRows / PJ_ROWS);
    rows_proj_tma_kernel<R, KR><<<grid, PJ_THREADS, C::SMEM, st>>>(a, c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles));
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// One adapter projection of a dense workspace tensor whose tensor map (box {64, 128}, 128-byte swizzle) is `map`.
tqp_status launch_rows_proj_tma(tqp_ctx *c, const CUtensorMap *map, int K, const bf16 *W, int w_kr, float s, bf16 *out, cudaStream_t st) {
    const int r = c->desc.r;
    ProjTmaArgs a;
    a.map = *map; a.W = W; a.out = out; a.K = K; a.s = s;
    if (r == 16 && w_kr) return launch_proj_tma_t<16, true>(c, a, st);
    if (r == 16) return launch_proj_tma_t<16, false>(c, a, st);
    if (r == 32 && w_kr) return launch_proj_tma_t<32, true>(c, a, st);
    if (r == 32) return launch_proj_tma_t<32, false>(c, a, st);
    return TQP_ERR_ARG;
}

// ---- gathered projections: rows by TMA gather4, write-through by TMA store -------------------------------------------
// Xp = gather(X) with x.A_g | x.A_u, and dYe = w . gather(dY) with dYe.B_d^T, for K % 256 == 0.
//
// What bounds the register-staged kernel above is not bytes but requests: it (and a first TMA version with 128-byte
// swizzled rows) moves the rows in 128-byte pieces and stays at ~2.6 TB/s.  A gather4 instruction costs the TMA unit the
// same ~70 clocks whether its four rows are 128 or 512 bytes wide, so this kernel gathers 256 columns (512 B) of a row
// at a time: a stage is 128 rows x 256 columns, DENSE (swizzling stops at 128-byte rows), 64 KB, three stages, one CTA
// per SM.  Warp 8 issues the gathers (lane l owns rows 4l..4l+3), warp 9 sends each landed stage to `through` (one
// tile store; a ragged last tile goes out with scatter4 so that the next expert's rows are never touched), warps 0-7
// multiply.
//
// Dense 512-byte rows put every row of one column in the same bank, which rules out ldmatrix for the row operand.  The
// A fragments are read with LDS.128 instead, in a PERMUTED k order: thread (g = lane/4, t = lane%4) takes the 16-byte
// chunks t and t+4 of every 64-column span of rows g and g+8 (odd g in the opposite order: the eight lanes of a
// quarter-warp then hit eight different bank groups), and feeds chunk words (0,1), (2,3) of chunk t to MMAs 0, 1 and
// those of chunk t+4 to MMAs 2, 3.  A sum over k does not care which physical column sits in which slot of the MMA as
// long as the adapter operand uses the same assignment: slot (2t+e) of MMA m holds column 32 (m/2) + 8t + 4 (m%2) + e,
// slot (8+2t+e) the column two further.  The adapter chunk is laid out in shared memory so that this read is
// conflict-free too: [R][K] matrices with a 96-element row (LDS.128 per thread), [K][R] matrices with ldmatrix.trans
// over hand-picked rows and a 32-byte skew every 8 rows.
// SCALE: the consumers first multiply their own 16 rows by the gate weight in place (bf16-rounded: the value the dH GEMM
// reads back), so the projection and the store both see the scaled rows.
constexpr int GP_THREADS = 320;   // 8 consumer warps, producer warp, store warp
constexpr int GP_COLS = 256;      // columns per stage
constexpr int GP_NST = 3;
template <int R, int NW, bool KR>
struct GatherCfg {
    static constexpr int RT = R * NW;
    static constexpr int WST = RT <= 32 ? 4 : 3;                      // adapter ring (64-k chunks)
    static constexpr int WLD = KR ? RT + 8 : 96;                      // KR: Ws[64][RT+8] (+16 elements every 8 rows), else Ws[RT][96]
    static constexpr int ROWS_BYTES = PJ_ROWS * GP_COLS * 2;          // 64 KB
    static constexpr int W_CHUNKS = KR ? PJ_KC * RT / 8 : RT * PJ_KC / 8;
    static constexpr int W_BYTES = KR ? PJ_KC * WLD * 2 + 256 : RT * WLD * 2;
    static constexpr int OFF_W = GP_NST * ROWS_BYTES;
    static constexpr int SMEM = OFF_W + WST * W_BYTES + 1024;
    static_assert(SMEM <= 232448, "shared memory");
};

struct GatherArgs {
    CUtensorMap in_map;    // source rows [in_rows][K], box {256, 1}, no swizzle (gather4)
    CUtensorMap out_map;   // through [out_rows][K], box {256, 128}, no swizzle (tile store)
    CUtensorMap sc_map;    // through, box {256, 1} (scatter4, ragged tiles)
    const int32_t *perm;   // row(p) = in[perm[p] / k]
    const float *roww;     // SCALE: row(p) *= roww[perm[p]]
    const bf16 *W[2];
    bf16 *out[2];
    int K, k, in_rows, out_rows;
    float s;
    int ablate;            // timing experiments only, as in ProjArgs: 256 no write-through, 512 no MMA
};

// One work item = 128 rows of one expert tile.  The kernel is persistent (one CTA per SM): the producer warp draws items
// from a global counter (whole 128-row halves of all tiles first, then the ragged second halves; item sizes differ a lot
// under skewed routing, so a fixed round-robin left SMs idle) and publishes each id in a small shared-memory queue that
// the store warp and the consumers follow.  Stage and adapter-ring counters run on across items, so the gathers of the
// next item are in flight while the consumers finish the current one.  Which CTA takes which item does not affect any
// result (items write disjoint rows).
struct GatherItem { int expert, row0, valid; };
constexpr int GP_QN = 8;   // item queue entries; the producer is at most GP_NST + 1 items ahead of its readers

template <int R, int NW, bool KR, bool SCALE>
__global__ void __launch_bounds__(GP_THREADS, 1) rows_gather_proj_kernel(const __grid_constant__ GatherArgs a, const Tile *__restrict__ tiles,
                                                                         const int32_t *__restrict__ num_tiles, int32_t *__restrict__ counter) {
    using C = GatherCfg<R, NW, KR>;
    using namespace ptx;
    constexpr int NST = GP_NST, WST = C::WST, HALVES = kTileRows / PJ_ROWS;
    __shared__ int s_q[GP_QN];   // published item ids (-1: no more)
    __shared__ int s_pub;        // number of entries published so far
    extern __shared__ uint8_t gp_smem_raw[];
    __shared__ __align__(8) uint64_t s_bar[3 * NST];   // full | empty | ready
    const int nt = *num_tiles, n_items = nt * HALVES;
    const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
    const uint32_t sbase = (smem_u32(gp_smem_raw) + 1023u) & ~1023u;
    const uint32_t full0 = smem_u32(s_bar), empty0 = full0 + 8 * NST, ready0 = full0 + 16 * NST;
    const int K = a.K, nst = K / GP_COLS, nq = K / PJ_KC;
    if (tid == 0) {
        s_pub = 0;
        for (int s = 0; s < NST; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, 9);    // 8 consumer warps + the store warp
            mbar_init(ready0 + 8 * s, 8);
        }
        mbar_init_fence();
    }
    __syncthreads();
    auto item = [&](int it) {   // item id -> rows; valid <= 0: nothing there (a tile of at most 128 rows has no second half)
        GatherItem g{0, 0, 0};
        if (it >= 0 && it < n_items) {
            const Tile t = tiles[it % nt];
            const int rbase = (it / nt) * PJ_ROWS;
            g.expert = t.expert; g.row0 = t.row0 + rbase; g.valid = min(PJ_ROWS, t.rows - rbase);
        }
        return g;
    };
    // the seq-th published item of this CTA (store warp and consumers; valid = 0: the queue has ended)
    auto published = [&](int seq) {
        while (*(volatile int *)&s_pub <= seq) {}
        __threadfence_block();
        return item(*(volatile int *)&s_q[seq % GP_QN]);
    };

    if (warp == 8) {   // ---- producer: gather4 of this lane's four rows, 256 columns per stage
        const uint64_t pol = l2_policy_evict_last();
        int n = 0;     // stages issued so far
        for (int seq = 0;; ++seq) {
            GatherItem g{0, 0, 0};
            int it = -1;
            do {   // draw until a non-empty item or the end
                if (lane == 0) it = atomicAdd(counter, 1);
                it = __shfl_sync(0xffffffffu, it, 0);
                g = item(it);
            } while (it < n_items && g.valid <= 0);
            if (lane == 0) {
                s_q[seq % GP_QN] = it < n_items ? it : -1;
                __threadfence_block();
                *(volatile int *)&s_pub = seq + 1;
            }
            if (it >= n_items) {   // no more work: the last CTA to get here re-arms the counters for the next launch (no memset node)
                if (lane == 0 && atomicAdd(counter + 1, 1) == (int)gridDim.x - 1) {
                    counter[0] = 0;
                    counter[1] = 0;
                }
                break;
            }
            const int nl = (g.valid + 3) / 4;
            int sr[4];     // rows past `valid`: an index past the tensor (zero fill, no traffic)
#pragma unroll
            for (int j = 0; j < 4; ++j) sr[j] = 4 * lane + j < g.valid ? a.perm[g.row0 + 4 * lane + j] / a.k : a.in_rows;
            for (int kc = 0; kc < nst; ++kc, ++n) {
                const int st = n % NST;
                if (n >= NST) mbar_wait(empty0 + 8 * st, ((n / NST) - 1) & 1);
                if (lane == 0) mbar_expect_tx(full0 + 8 * st, nl * 4 * GP_COLS * 2);
                __syncwarp();
                if (lane < nl)
                    tma_gather4(sbase + st * C::ROWS_BYTES + lane * (4 * GP_COLS * 2), &a.in_map, kc * GP_COLS, sr[0], sr[1], sr[2], sr[3],
                                full0 + 8 * st, pol);
            }
        }
        return;
    }
    if (warp == 9) {   // ---- store: stage -> through[row0 .. row0 + valid)
        const uint64_t pol = l2_policy_evict_first();
        int n = 0;
        for (int seq = 0;; ++seq) {
            const GatherItem g = published(seq);
            if (g.valid <= 0) break;
            const int nl = (g.valid + 3) / 4;
            int dr[4];     // ragged tile: rows past `valid` get an index past the tensor (clipped, never written)
#pragma unroll
            for (int j = 0; j < 4; ++j) dr[j] = 4 * lane + j < g.valid ? g.row0 + 4 * lane + j : a.out_rows;
            const bool whole = g.valid == PJ_ROWS;
            for (int kc = 0; kc < nst; ++kc, ++n) {
                const int st = n % NST;
                mbar_wait((SCALE ? ready0 : full0) + 8 * st, (n / NST) & 1);
                const uint32_t rows_s = sbase + st * C::ROWS_BYTES;
                if (!TQP_DBG(a.ablate & 256) && (whole ? lane == 0 : lane < nl)) {
                    if (whole) tma_store_2d(&a.out_map, kc * GP_COLS, g.row0, rows_s, pol);
                    else tma_scatter4(&a.sc_map, kc * GP_COLS, dr[0], dr[1], dr[2], dr[3], rows_s + lane * (4 * GP_COLS * 2), pol);
                    bulk_commit_group();
                    bulk_wait_group_read<0>();   // the stage has been read: it may be refilled
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty0 + 8 * st);
            }
        }
        return;
    }

    // ---- consumers (256 threads): adapter chunks by cp.async, MMAs on the gathered rows
    auto issue_w = [&](int expert, int q, int slot) {   // 64-k adapter chunk q of `expert` -> ring slot
        const uint32_t w_s = sbase + C::OFF_W + slot * C::W_BYTES;
        for (int v = tid; v < C::W_CHUNKS; v += PJ_THREADS) {
            if (KR) {   // W_w[e][k][R] -> Ws[k][w R + q], rows skewed by 16 elements every 8
                const int kk = v / (C::RT / 8), cc = v % (C::RT / 8), w = (cc * 8) / R, q0 = (cc * 8) % R;
                cp_async16(w_s + (kk * C::WLD + (kk / 8) * 16 + cc * 8) * 2, a.W[w] + ((size_t)expert * K + q * PJ_KC + kk) * R + q0, 16);
            } else {    // W_w[e][q][K] -> Ws[w R + q][k]
                const int n = v / (PJ_KC / 8), cc = v % (PJ_KC / 8), w = n / R, qq = n % R;
                cp_async16(w_s + (n * C::WLD + cc * 8) * 2, a.W[w] + ((size_t)expert * R + qq) * K + q * PJ_KC + cc * 8, 16);
            }
        }
    };
    const int g8 = lane >> 2, tq = lane & 3, odd = g8 & 1;
    const uint32_t a_off = (warp * 16 + g8) * (GP_COLS * 2) + (tq + 4 * odd) * 16;   // first chunk of this lane in a span
    const int a_sw = odd ? -64 : 64;                                                 // byte offset of its second chunk
    // [K][R] adapters: lane (i = lane%8, j = (lane/8)%2, nb = lane/16) addresses row 8 (i/2) + i%2 + 2 j of the chunk
    const int li = lane & 7, lj = (lane >> 3) & 1;
    const int kl = 8 * (li >> 1) + (li & 1) + 2 * lj;
    const uint32_t bk_off = (kl * C::WLD + (li >> 1) * 16 + (lane >> 4) * 8) * 2;
    const uint32_t bn_off = (g8 * C::WLD + 8 * tq) * 2;                               // [R][K] adapters

    int seq = 0;
    GatherItem cur = published(seq);
    int n = 0, wq = 0;   // stages / adapter chunks consumed so far
    if (cur.valid > 0)
        for (int s = 0; s < WST - 1; ++s) { issue_w(cur.expert, s, s); cp_async_commit(); }   // nq >= 4 > WST - 1
    while (cur.valid > 0) {
        GatherItem nxt{0, 0, 0};
        bool have_nxt = false;   // looked up when the adapter ring first reaches past this item: by then the producer has
                                 // issued this item's last stage and is drawing the next
        float acc[C::RT / 8][4];
#pragma unroll
        for (int i = 0; i < C::RT / 8; ++i)
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[i][q] = 0.f;
        const bool active = warp * 16 < cur.valid;
        float roww = 1.f;   // SCALE: lane l (< 16) holds the gate weight of row 16 warp + l
        if (SCALE && lane < 16 && warp * 16 + lane < cur.valid) roww = a.roww[a.perm[cur.row0 + warp * 16 + lane]];
        for (int q = 0; q < nq; ++q, ++wq) {
            const int ss = q % 4, st = n % NST;
            const uint32_t rows_s = sbase + st * C::ROWS_BYTES, w_s = sbase + C::OFF_W + (wq % WST) * C::W_BYTES;
            cp_async_wait<WST - 2>();
            named_bar_sync(1, PJ_THREADS);   // adapter chunk wq visible; every consumer is past the MMAs of chunk wq - 1
            {   // refill the slot chunk wq - 1 used: the chunk WST - 1 ahead, of this item or the first of the next
                const int qa = q + WST - 1, slot = (wq + WST - 1) % WST;
                if (qa < nq) issue_w(cur.expert, qa, slot);
                else {
                    if (!have_nxt) { nxt = published(seq + 1); have_nxt = true; }
                    if (nxt.valid > 0) issue_w(nxt.expert, qa - nq, slot);
                }
                cp_async_commit();
            }
            if (ss == 0) {
                mbar_wait(full0 + 8 * st, (n / NST) & 1);
                if (SCALE) {
                    if (active) {
                        const uint32_t mine = rows_s + warp * 16 * (GP_COLS * 2) + lane * 16;
#pragma unroll 4
                        for (int i = 0; i < 16; ++i) {   // row 16 warp + i: 32 lanes x 16 bytes
                            const float wr = __shfl_sync(0xffffffffu, roww, i);
                            uint4 v = lds128(mine + i * (GP_COLS * 2));
                            uint32_t *vp = reinterpret_cast<uint32_t *>(&v);
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const float2 f = bf16x2_to_float2(vp[e]);
                                vp[e] = float2_to_bf16x2(wr * f.x, wr * f.y);
                            }
                            sts128(mine + i * (GP_COLS * 2), v);
                        }
                        fence_async_smem();   // the TMA store (async proxy) must see the scaled rows
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(ready0 + 8 * st);
                }
            }
            if (active && !TQP_DBG(a.ablate & 512)) {
                const uint32_t ra = rows_s + a_off + ss * 128;
                const uint4 x0 = lds128(ra), x1 = lds128(ra + a_sw), y0 = lds128(ra + 8 * GP_COLS * 2), y1 = lds128(ra + 8 * GP_COLS * 2 + a_sw);
                const uint4 P = odd ? x1 : x0, Q = odd ? x0 : x1, P8 = odd ? y1 : y0, Q8 = odd ? y0 : y1;   // chunk t | t+4 of rows g | g+8
                const uint32_t af[4][4] = {{P.x, P8.x, P.y, P8.y}, {P.z, P8.z, P.w, P8.w}, {Q.x, Q8.x, Q.y, Q8.y}, {Q.z, Q8.z, Q.w, Q8.w}};
                if (KR) {
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        const uint32_t bm = w_s + bk_off + ((32 * (m / 2) + 4 * (m % 2)) * C::WLD + 4 * (m / 2) * 16) * 2;
#pragma unroll
                        for (int np = 0; np < C::RT / 16; ++np) {
                            uint32_t bq[4];
                            ldsm_x4_t(bm + np * 32, bq);
                            mma16816(acc[2 * np], af[m], bq[0], bq[1]);
                            mma16816(acc[2 * np + 1], af[m], bq[2], bq[3]);
                        }
                    }
                } else {
#pragma unroll
                    for (int nb = 0; nb < C::RT / 8; ++nb) {
                        const uint4 w0 = lds128(w_s + bn_off + nb * 8 * C::WLD * 2), w1 = lds128(w_s + bn_off + nb * 8 * C::WLD * 2 + 64);
                        mma16816(acc[nb], af[0], w0.x, w0.y);
                        mma16816(acc[nb], af[1], w0.z, w0.w);
                        mma16816(acc[nb], af[2], w1.x, w1.y);
                        mma16816(acc[nb], af[3], w1.z, w1.w);
                    }
                }
            }
            if (ss == 3) {
                __syncwarp();
                if (lane == 0) mbar_arrive(empty0 + 8 * st);
                ++n;
            }
        }
        if (active) {
#pragma unroll
            for (int i = 0; i < C::RT / 8; ++i) {
                const int col = i * 8 + (lane % 4) * 2, w = col / R, q = col % R;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int r = warp * 16 + lane / 4 + 8 * h;
                    if (r < cur.valid)
                        *reinterpret_cast<uint32_t *>(a.out[w] + (size_t)(cur.row0 + r) * kLoraPad + q) =
                            float2_to_bf16x2(a.s * acc[i][2 * h], a.s * acc[i][2 * h + 1]);
                }
            }
        }
        cur = nxt;   // nq >= WST - 1 chunks: the look-up above has happened
        ++seq;
    }
    cp_async_wait<0>();
}

template <int R, int NW, bool KR, bool SCALE>
static tqp_status launch_gather_t(tqp_ctx *c, const GatherArgs &a, cudaStream_t st) {
    using C = GatherCfg<R, NW, KR>;
    if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&rows_gather_proj_kernel<R, NW, KR, SCALE>), C::SMEM)) return st_attr;
    const int grid = std::min(c->num_sms, c->max_tiles * (kTileRows / PJ_ROWS));
    int32_t *counter = c->p<int32_t>(c->ws.sched);   // [0] items drawn, [1] CTAs finished: zero at bind, re-armed by the kernel
    rows_gather_proj_kernel<R, NW, KR, SCALE><<<grid, GP_THREADS, C::SMEM, st>>>(a, c->p<Tile>(c->ws.tiles), c->p<int32_t>(c->ws.num_tiles), counter);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// through[p] = (roww ? roww[perm[p]] : 1) . in[perm[p] / k]  and  out_w[p] = s . through[p] . W_w[e(p)]   (r = 16 / 32,
// K % 256 == 0).  Unswizzled maps: in_map = the source with box {256, 1}; out_map / sc_map = `through` with box
// {256, 128} / {256, 1}.
tqp_status launch_rows_gather_proj(tqp_ctx *c, const CUtensorMap *in_map, int in_rows, const CUtensorMap *out_map, const CUtensorMap *sc_map,
                                   int out_rows, int K, const int32_t *perm, const float *roww, const bf16 *W0, const bf16 *W1, int w_kr,
                                   float s, bf16 *out0, bf16 *out1, cudaStream_t st) {
    const int r = c->desc.r;
    GatherArgs a;
    a.in_map = *in_map; a.out_map = *out_map; a.sc_map = *sc_map; a.perm = perm; a.roww = roww;
    a.W[0] = W0; a.W[1] = W1; a.out[0] = out0; a.out[1] = out1; a.K = K; a.k = c->desc.k; a.in_rows = in_rows; a.out_rows = out_rows; a.s = s; a.ablate = c->ablate;
    const bool kr = w_kr != 0, two = W1 != nullptr, sc = roww != nullptr;
    if (K % GP_COLS) return TQP_ERR_ARG;
    // the two shapes the layer uses: x.A_g | x.A_u (two [K][R] matrices, no scale) and w dY . B_d^T (one [R][K] matrix, scaled)
    if (r == 16 && two && kr && !sc) return launch_gather_t<16, 2, true, false>(c, a, st);
    if (r == 32 && two && kr && !sc) return launch_gather_t<32, 2, true, false>(c, a, st);
    if (r == 16 && !two && !kr && sc) return launch_gather_t<16, 1, false, true>(c, a, st);
    if (r == 32 && !two && !kr && sc) return launch_gather_t<32, 1, false, true>(c, a, st);
    return TQP_ERR_ARG;
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

// nw projections of the same rows in one pass.  perm/roww/through select the gathered (fused dispatch / combine-bwd)
// variants; rank 8 (config 0) runs on CUDA cores from an already dense `in`.
tqp_status launch_rows_proj(tqp_ctx *c, const bf16 *in, int K, const int32_t *perm, const float *roww, bf16 *through,
                            const bf16 *W0, const bf16 *W1, int w_kr, float s, bf16 *out0, bf16 *out1, cudaStream_t st) {
    const int r = c->desc.r, nw = W1 ? 2 : 1;
    if (r != 16 && r != 32) {
        if (perm || roww || through) { c->err = "rows_proj: gathered variants need r = 16 or 32"; return TQP_ERR_ARG; }
        const Tile *tiles = c->p<Tile>(c->ws.tiles);
        const int32_t *nt = c->p<int32_t>(c->ws.num_tiles);
        dim3 grid(c->max_tiles, kTileRows / 64);
        lora_down_small_kernel<<<grid, 128, 0, st>>>(in, K, r, W0, w_kr, s, out0, tiles, nt);
        TQP_LAUNCH_OK(c);
        if (W1) {
            lora_down_small_kernel<<<grid, 128, 0, st>>>(in, K, r, W1, w_kr, s, out1, tiles, nt);
            TQP_LAUNCH_OK(c);
        }
        return TQP_OK;
    }
    ProjArgs a;
    a.in = in; a.perm = perm; a.roww = roww; a.through = through; a.W[0] = W0; a.W[1] = W1; a.out[0] = out0; a.out[1] = out1;
    a.K = K; a.k = c->desc.k; a.s = s; a.ablate = c->ablate;
#define TQP_PJ(R_, NW_, KR_) if (r == R_ && nw == NW_ && (w_kr != 0) == KR_) return launch_proj_t<R_, NW_, KR_>(c, a, st)
    TQP_PJ(16, 1, true); TQP_PJ(16, 2, true); TQP_PJ(16, 1, false); TQP_PJ(16, 2, false);
    TQP_PJ(32, 1, true); TQP_PJ(32, 2, true); TQP_PJ(32, 1, false); TQP_PJ(32, 2, false);
#undef TQP_PJ
    return TQP_ERR_ARG;
}

// ---- weight gradients -------------------------------------------------------------------------------------------
constexpr int WG_ROWS = 32;             // rows per stage
constexpr int WG_COLS = 128;            // columns of `big` per CTA (4 warps x 32)
constexpr int WG_LD = WG_COLS + 8;
constexpr int WG_NST = 4;

struct WgradArgs {
    const bf16 *big;         // [N][width]
    const bf16 *small_[2];   // [N][kLoraPad]
    float *grad[2];          // out_ar: [E][width][R] (dA) else [E][R][width] (dB)
    int width, out_ar;
    // experts with more than kWgradSeg rows are split into row segments (one CTA each); their partial gradients go to
    // `scratch` (entry e: first segment of expert e; entry E + j: extra segment j of the device-built list) and are
    // summed in segment order by the CTA that finishes last -- deterministic, no atomics on the data
    const Tile *xsegs;
    const int32_t *xfirst;   // [E + 1]: first extra segment of every expert; xfirst[E] = number of extra segments
    float *scratch;
    int E;
    size_t entry;            // floats per scratch entry = ns * R * width
    int32_t *done;           // [E][width / 128] arrival counters of split experts (zero between launches: the last arriver resets its own)
};

template <int R, int NS>
struct WgradCfg {
    static constexpr int RT = R * NS;
    static constexpr int SLD = RT + 8;
    static constexpr int BIG_BYTES = WG_ROWS * WG_LD * 2;
    static constexpr int SM_BYTES = (WG_ROWS * SLD * 2 + 127) / 128 * 128;
    static constexpr int STAGE = BIG_BYTES + SM_BYTES;
    static constexpr int SMEM = WG_NST * STAGE + 128;
};

// grid = (E + max extra segments) x (width / 128) CTAs, block = 128.  Warp w owns columns [32 w, 32 w + 32) of the slab and all RT
// adapter columns.  Blocks [0, E): the first kWgradSeg rows of expert blockIdx.x; blocks >= E: one extra segment each.
template <int R, int NS>
__global__ void __launch_bounds__(128) rows_wgrad_kernel(const __grid_constant__ WgradArgs a, const int32_t *__restrict__ offsets) {
    using C = WgradCfg<R, NS>;
    extern __shared__ __align__(128) uint8_t wg_smem[];
    uint8_t *smem = wg_smem;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    // 1-D grid, slab index fastest: the column slabs of one expert run side by side, so that the 256-byte pieces they take
    // from the same rows arrive at the DRAM pages together
    const int nslab = a.width / WG_COLS, bx = blockIdx.x / nslab;
    const int a0 = (blockIdx.x % nslab) * WG_COLS;
    const int tid = threadIdx.x, warp = tid / 32;
    const int width = a.width;
    int e, p0, p1;
    float *dst[2];
    bool split;   // the expert has more than kWgradSeg rows: this CTA writes a partial, the last CTA of the expert's slab sums them
    if (bx < a.E) {
        e = bx;
        p0 = offsets[e];
        const int cnt = offsets[e + 1] - p0;
        p1 = p0 + min(cnt, kWgradSeg);
        split = cnt > kWgradSeg;
#pragma unroll
        for (int w = 0; w < NS; ++w)
            dst[w] = split ? a.scratch + (size_t)e * a.entry + (size_t)w * R * width : a.grad[w] + (size_t)e * R * width;
    } else {
        const int j = bx - a.E;
        if (j >= a.xfirst[a.E]) return;
        const Tile t = a.xsegs[j];
        e = t.expert;
        p0 = t.row0;
        p1 = p0 + t.rows;
        split = true;
#pragma unroll
        for (int w = 0; w < NS; ++w) dst[w] = a.scratch + (size_t)(a.E + j) * a.entry + (size_t)w * R * width;
    }
    const int nit = (p1 - p0 + WG_ROWS - 1) / WG_ROWS;

    auto issue = [&](int it, int st) {
        const int p = p0 + it * WG_ROWS;
        const uint32_t big_s = sbase + st * C::STAGE, sm_s = big_s + C::BIG_BYTES;
        // rows at or past p1 belong to the next expert: zero-filled (src-size 0), address clamped to a valid row
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int r = tid / 16 + 8 * i, cc = tid % 16;
            const bool ok = p + r < p1;
            cp_async16(big_s + (r * WG_LD + cc * 8) * 2, a.big + (size_t)(ok ? p + r : p1 - 1) * width + a0 + cc * 8, ok ? 16 : 0);
        }
        for (int v = tid; v < WG_ROWS * C::RT / 8; v += 128) {
            const int r = v / (C::RT / 8), cc = v % (C::RT / 8), w = (cc * 8) / R, q0 = (cc * 8) % R;
            const bool ok = p + r < p1;
            cp_async16(sm_s + (r * C::SLD + cc * 8) * 2, a.small_[w] + (size_t)(ok ? p + r : p1 - 1) * kLoraPad + q0, ok ? 16 : 0);
        }
    };

    float acc[C::RT / 16][4][4];   // [16 adapter columns][8 big columns][fragment]
#pragma unroll
    for (int m = 0; m < C::RT / 16; ++m)
#pragma unroll
        for (int n = 0; n < 4; ++n)
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[m][n][q] = 0.f;
    const int lane = tid % 32;
    for (int s = 0; s < WG_NST - 1; ++s) {
        if (s < nit) issue(s, s);
        cp_async_commit();
    }
    // A = small^T (stored [p][q]) and B = big (stored [p][a]) are both read with ldmatrix.trans
    const uint32_t a_off = (((lane / 16) * 8 + lane % 8) * C::SLD + ((lane / 8) % 2) * 8) * 2;
    const uint32_t b_off = ((((lane / 8) % 2) * 8 + lane % 8) * WG_LD + warp * 32 + (lane / 16) * 8) * 2;
    for (int it = 0; it < nit; ++it) {
        const int st = it % WG_NST;
        cp_async_wait<WG_NST - 2>();
        __syncthreads();
        if (it + WG_NST - 1 < nit) issue(it + WG_NST - 1, (it + WG_NST - 1) % WG_NST);
        cp_async_commit();
        const uint32_t big_s = sbase + st * C::STAGE, sm_s = big_s + C::BIG_BYTES;
#pragma unroll
        for (int pp = 0; pp < WG_ROWS; pp += 16) {
            uint32_t af[C::RT / 16][4];
#pragma unroll
            for (int m = 0; m < C::RT / 16; ++m) ldsm_x4_t(sm_s + a_off + (pp * C::SLD + m * 16) * 2, af[m]);
#pragma unroll
            for (int np = 0; np < 2; ++np) {
                uint32_t bq[4];
                ldsm_x4_t(big_s + b_off + (pp * WG_LD + np * 16) * 2, bq);
#pragma unroll
                for (int m = 0; m < C::RT / 16; ++m) {
                    mma16816(acc[m][2 * np], af[m], bq[0], bq[1]);
                    mma16816(acc[m][2 * np + 1], af[m], bq[2], bq[3]);
                }
            }
        }
    }
    cp_async_wait<0>();
#pragma unroll
    for (int m = 0; m < C::RT / 16; ++m) {
        const int w = (m * 16) / R;
#pragma unroll
        for (int n = 0; n < 4; ++n) {
            const int col = a0 + warp * 32 + n * 8 + (lane % 4) * 2;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int q = (m * 16) % R + lane / 4 + 8 * h;
                if (a.out_ar) {   // [col][q]
                    float *g = dst[w] + (size_t)col * R + q;
                    g[0] = acc[m][n][2 * h];
                    g[R] = acc[m][n][2 * h + 1];
                } else {          // [q][col]
                    *reinterpret_cast<float2 *>(dst[w] + (size_t)q * width + col) =
                        make_float2(acc[m][n][2 * h], acc[m][n][2 * h + 1]);
                }
            }
        }
    }
    if (!split) return;
    // Split expert: the CTA that arrives last at the expert's slab counter sums the partials of this slab in SEGMENT order (first
    // segment, then the extra segments of the device-built list) -- deterministic whoever arrives last, no atomics on the data --
    // and resets the counter for the next launch.  (A separate reduction kernel per gradient cost 4 us + a launch gap even when no
    // expert was split, 10-46 us under skew.)
    __shared__ int s_last;
    const int x0 = a.xfirst[e], nx = a.xfirst[e + 1] - x0;
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        int32_t *cnt = a.done + (size_t)e * nslab + a0 / WG_COLS;
        const int prev = atomicAdd(cnt, 1);
        s_last = prev == nx;
        if (prev == nx) *cnt = 0;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
#pragma unroll
    for (int w = 0; w < NS; ++w) {
        const float *first = a.scratch + (size_t)e * a.entry + (size_t)w * R * width;
        float *out = a.grad[w] + (size_t)e * R * width;
        // this slab's region: out_ar ? rows [a0, a0 + 128) of [width][R] (contiguous) : columns [a0, a0 + 128) of each of the R rows
        for (int v = tid; v < R * WG_COLS / 4; v += 128) {
            const size_t off = a.out_ar ? (size_t)a0 * R + (size_t)v * 4 : (size_t)(v / (WG_COLS / 4)) * width + a0 + (v % (WG_COLS / 4)) * 4;
            float4 sum = __ldcg(reinterpret_cast<const float4 *>(first + off));
            for (int j = 0; j < nx; ++j) {
                const float4 t4 = __ldcg(reinterpret_cast<const float4 *>(a.scratch + (size_t)(a.E + x0 + j) * a.entry + (size_t)w * R * width + off));
                sum.x += t4.x; sum.y += t4.y; sum.z += t4.z; sum.w += t4.w;
            }
            *reinterpret_cast<float4 *>(out + off) = sum;
        }
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

template <int R, int NS>
static tqp_status launch_wgrad_t(tqp_ctx *c, const WgradArgs &a, const int32_t *offsets, cudaStream_t st) {
    using C = WgradCfg<R, NS>;
    if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&rows_wgrad_kernel<R, NS>), C::SMEM)) return st_attr;
    rows_wgrad_kernel<R, NS><<<(unsigned)((c->desc.E + c->max_xsegs) * (a.width / WG_COLS)), 128, C::SMEM, st>>>(a, offsets);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// ns weight gradients that share the streamed operand `big` (e.g. dA_gate and dA_up both contract Xp) in one pass.
tqp_status launch_rows_wgrad(tqp_ctx *c, const bf16 *big, int width, const bf16 *small0, const bf16 *small1,
                             const int32_t *offsets, int out_ar, float *grad0, float *grad1, cudaStream_t st) {
    const int r = c->desc.r, E = c->desc.E;
    if (r != 16 && r != 32) {
        lora_wgrad_small_kernel<<<dim3(E, 8), 256, 0, st>>>(big, width, r, small0, offsets, out_ar, grad0);
        TQP_LAUNCH_OK(c);
        if (small1) {
            lora_wgrad_small_kernel<<<dim3(E, 8), 256, 0, st>>>(big, width, r, small1, offsets, out_ar, grad1);
            TQP_LAUNCH_OK(c);
        }
        return TQP_OK;
    }
    WgradArgs a;
    a.big = big; a.small_[0] = small0; a.small_[1] = small1; a.grad[0] = grad0; a.grad[1] = grad1;
    a.width = width; a.out_ar = out_ar;
    const int ns = small1 ? 2 : 1;
    a.xsegs = c->p<Tile>(c->ws.xsegs); a.xfirst = c->p<int32_t>(c->ws.xfirst); a.scratch = c->p<float>(c->ws.wg_scratch);
    a.E = E; a.entry = (size_t)ns * r * width; a.done = c->p<int32_t>(c->ws.wg_done);
    if (r == 16 && ns == 1) return launch_wgrad_t<16, 1>(c, a, offsets, st);
    if (r == 16 && ns == 2) return launch_wgrad_t<16, 2>(c, a, offsets, st);
    if (r == 32 && ns == 1) return launch_wgrad_t<32, 1>(c, a, offsets, st);
    return launch_wgrad_t<32, 2>(c, a, offsets, st);
}

// ---- dG . B_g^T | dU . B_u^T together with (x.A_g)^T dG | (x.A_u)^T dU: one pass over dG and dU -----------------------------
// The backward of the gate / up adapters needs dG (and dU) twice: the projection Z = s dG . B^T (the adapter K-step of the dXp
// GEMM and the row operand of dA) and the weight gradient dB = (s x.A)^T dG.  As separate passes (rows_proj_tma + rows_wgrad)
// each streams the [N][F] tensor from HBM; here one CTA owns one grouped-GEMM tile (<= 256 rows of one expert), streams its
// rows once in 64-column TMA stages (the GEMM's own tensor map: box {64, 256}, 128-byte swizzle) and feeds both
// contractions from the stage: warp w multiplies rows [32 w, 32 w + 32) by the adapter chunk (projection, accumulated over
// the whole width) and columns [8 w, 8 w + 8) of the stage by the tile's x.A rows (weight gradient: complete for this tile
// after every stage, written out and reset).  An expert with one tile writes its gradient directly; an expert with several
// writes per-tile partials to the scratch and projwg_reduce_kernel sums them in tile order (deterministic, no atomics);
// experts without rows are zeroed there.  grid = (max_tiles, 2): y = 0 gate, 1 up.  (Loading only the 32-row boxes that hold rows
// of the tile instead of one 256-row box reads 12 % fewer bytes at cfg 2 but was slower, 117 against 107 us: seven TMA
// instructions per stage from one thread.)
template <int R>
struct ProjWgCfg {
    static constexpr int NST = R == 16 ? 3 : 2;                       // 112 KB (r = 16) / 90 KB (r = 32): two CTAs per SM                       // r = 16: 112 KB, two CTAs per SM (one CTA with six stages: 129 against 106 us at cfg 2)
    static constexpr int WLD = PJ_LD;                                 // adapter chunk Ws[R][64 + 8]
    static constexpr int ROWS_BYTES = kTileRows * PJ_KC * 2;          // 32 KB (swizzled, unpadded)
    static constexpr int W_BYTES = (R * WLD * 2 + 127) / 128 * 128;
    static constexpr int CPR = R / 8;                                 // 16-byte chunks per x.A row
    static constexpr int S_BYTES = kTileRows * R * 2;                 // x.A rows of the tile, dense [256][R], chunks XOR-swizzled
    static constexpr int OFF_W = NST * ROWS_BYTES;
    static constexpr int OFF_S = OFF_W + NST * W_BYTES;
    static constexpr int SMEM = OFF_S + S_BYTES + 1024;
};

struct ProjWgArgs {
    CUtensorMap map[2];      // dG, dU: [N][F], box {64, 256}, SWIZZLE_128B
    const bf16 *W[2];        // B_gate, B_up: [E][R][F]
    const bf16 *small_[2];   // s x.A_g, s x.A_u: [N][kLoraPad]
    bf16 *out[2];            // Z_g, Z_u: [N][kLoraPad]
    float *grad[2];          // dB_gate, dB_up: [E][R][F]
    float *scratch;          // [2][max_tiles][R][F] partials of experts with more than one tile
    const int32_t *tfirst;   // [E + 1]: expert e owns tiles [tfirst[e], tfirst[e + 1])
    int K, E, max_tiles;
    float s;
};

template <int R>
__global__ void __launch_bounds__(PJ_THREADS, 2) rows_proj_wgrad_kernel(const __grid_constant__ ProjWgArgs a,
                                                                                      const Tile *__restrict__ tiles,
                                                                                      const int32_t *__restrict__ num_tiles) {
    using C = ProjWgCfg<R>;
    using namespace ptx;
    constexpr int NST = C::NST, MT = R / 16;
    extern __shared__ uint8_t pw_smem_raw[];
    __shared__ __align__(8) uint64_t s_full[NST];
    const int nt_all = *num_tiles, j = blockIdx.x, y = blockIdx.y;
    if (j >= nt_all) return;
    const Tile t = tiles[j];
    const int valid = t.rows, row0 = t.row0, e = t.expert;
    if (valid <= 0) return;
    const bool single = (j == 0 || tiles[j - 1].expert != e) && (j + 1 >= nt_all || tiles[j + 1].expert != e);
    const int K = a.K, nk = K / PJ_KC;
    float *dst = single ? a.grad[y] + (size_t)e * R * K : a.scratch + ((size_t)y * a.max_tiles + j) * R * K;
    const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
    const uint32_t sbase = (smem_u32(pw_smem_raw) + 1023u) & ~1023u;
    const uint32_t bar0 = smem_u32(s_full), s_s = sbase + C::OFF_S;
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_init_fence();
    }
    __syncthreads();
    const CUtensorMap *map = &a.map[y];
    const bf16 *W = a.W[y] + (size_t)e * R * K;
    auto issue = [&](int kc) {   // rows by TMA (one thread), adapter chunk by cp.async (everyone)
        const int st = kc % NST;
        if (tid == 0) {
            mbar_expect_tx(bar0 + 8 * st, C::ROWS_BYTES);
            tma_load_2d(sbase + st * C::ROWS_BYTES, map, kc * PJ_KC, row0, bar0 + 8 * st);
        }
        const uint32_t w_s = sbase + C::OFF_W + st * C::W_BYTES;
        for (int v = tid; v < R * PJ_KC / 8; v += PJ_THREADS) {
            const int q = v / (PJ_KC / 8), cc = v % (PJ_KC / 8);
            cp_async16(w_s + (q * C::WLD + cc * 8) * 2, W + (size_t)q * K + kc * PJ_KC + cc * 8, 16);
        }
    };
    // the tile's x.A rows (zero past `valid`: those stage rows belong to the next tile); part of the first commit group
    for (int v = tid; v < kTileRows * C::CPR; v += PJ_THREADS) {
        const int pr = v / C::CPR, cc = v % C::CPR;
        const bool ok = pr < valid;
        cp_async16(s_s + pr * (R * 2) + ((cc ^ ((pr * C::CPR / 8) % C::CPR)) << 4), a.small_[y] + (size_t)(row0 + (ok ? pr : 0)) * kLoraPad + cc * 8,
                   ok ? 16 : 0);
    }
    for (int s = 0; s < NST - 1; ++s) {
        if (s < nk) issue(s);
        cp_async_commit();
    }
    float acc[2][R / 8][4], wacc[MT][4];
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int n = 0; n < R / 8; ++n)
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[m][n][q] = 0.f;
#pragma unroll
    for (int m = 0; m < MT; ++m)
#pragma unroll
        for (int q = 0; q < 4; ++q) wacc[m][q] = 0.f;
    const int prow = warp * 32 + lane % 16;   // this lane's row of the projection's A fragments (ldmatrix x4), first 16-row group
    for (int kc = 0; kc < nk; ++kc) {
        const int st = kc % NST;
        mbar_wait(bar0 + 8 * st, (kc / NST) & 1);
        cp_async_wait<NST - 2>();
        __syncthreads();   // chunk kc visible to everyone; everyone is past chunk kc - 1 (its stage is refilled below)
        if (kc + NST - 1 < nk) issue(kc + NST - 1);
        cp_async_commit();
        const uint32_t rows_s = sbase + st * C::ROWS_BYTES, w_s = sbase + C::OFF_W + st * C::W_BYTES;
        // projection: rows [32 warp, 32 warp + 32) x this 64-column chunk of the adapter
        if (warp * 32 < valid) {
            const uint32_t b_addr = w_s + (((lane / 16) * 8 + lane % 8) * C::WLD + ((lane / 8) % 2) * 8) * 2;
#pragma unroll
            for (int kk = 0; kk < PJ_KC; kk += 16) {
                uint32_t bq[MT][4];
#pragma unroll
                for (int np = 0; np < MT; ++np) ldsm_x4(b_addr + (np * 16 * C::WLD + kk) * 2, bq[np]);
#pragma unroll
                for (int m = 0; m < 2; ++m) {
                    if (warp * 32 + 16 * m >= valid) continue;
                    const int ar = prow + 16 * m;
                    uint32_t af[4];
                    ldsm_x4(rows_s + ar * 128 + ((((kk >> 3) + (lane >> 4)) ^ (ar & 7)) << 4), af);
#pragma unroll
                    for (int np = 0; np < MT; ++np) {
                        mma16816(acc[m][2 * np], af, bq[np][0], bq[np][1]);
                        mma16816(acc[m][2 * np + 1], af, bq[np][2], bq[np][3]);
                    }
                }
            }
        }
        // weight gradient: (x.A)^T [R x rows] . stage [rows x 8 columns of this warp], two 16-row k-steps per load
        for (int pb = 0; pb < valid; pb += 32) {
            uint32_t bq[4];
            const int pr = pb + lane;
            ldsm_x4_t(rows_s + pr * 128 + ((warp ^ (pr & 7)) << 4), bq);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int pa = pb + 16 * h + (lane / 16) * 8 + lane % 8;
#pragma unroll
                for (int m = 0; m < MT; ++m) {
                    uint32_t af[4];
                    const int cq = 2 * m + (lane / 8) % 2;
                    ldsm_x4_t(s_s + pa * (R * 2) + ((cq ^ ((pa * C::CPR / 8) % C::CPR)) << 4), af);
                    mma16816(wacc[m], af, bq[2 * h], bq[2 * h + 1]);
                }
            }
        }
        {
            const int col = kc * PJ_KC + warp * 8 + (lane % 4) * 2;
#pragma unroll
            for (int m = 0; m < MT; ++m) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    *reinterpret_cast<float2 *>(dst + (size_t)(m * 16 + lane / 4 + 8 * h) * K + col) = make_float2(wacc[m][2 * h], wacc[m][2 * h + 1]);
                    wacc[m][2 * h] = 0.f;
                    wacc[m][2 * h + 1] = 0.f;
                }
            }
        }
    }
    cp_async_wait<0>();
#pragma unroll
    for (int m = 0; m < 2; ++m) {
#pragma unroll
        for (int n = 0; n < R / 8; ++n) {
            const int q = n * 8 + (lane % 4) * 2;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = warp * 32 + 16 * m + lane / 4 + 8 * h;
                if (r < valid)
                    *reinterpret_cast<uint32_t *>(a.out[y] + (size_t)(row0 + r) * kLoraPad + q) =
                        float2_to_bf16x2(a.s * acc[m][n][2 * h], a.s * acc[m][n][2 * h + 1]);
            }
        }
    }
}

// grid = (E, 2, PWR_SPLIT), block = 256: expert e, gate / up, one slice of the [R][F] gradient.  No tile: the slice is zeroed; one tile: nothing to do (the kernel wrote the
// gradient itself); several: their partials are summed in tile order.  (One CTA per expert was 200 us at cfg 3, where one
// expert owns dozens of tiles.)
constexpr int PWR_SPLIT = 8;
__global__ void __launch_bounds__(256) projwg_reduce_kernel(const __grid_constant__ ProjWgArgs a, const Tile *__restrict__ tiles, int R) {
    const int e = blockIdx.x, y = blockIdx.y;
    const size_t per = (size_t)R * a.K, slice = per / 4 / PWR_SPLIT;   // float4 elements; R F / 4 is a multiple of 8 (F % 64 == 0)
    const int j = a.tfirst[e], n = a.tfirst[e + 1] - j;   // the expert's tiles (dispatch)
    if (n == 1) return;
    float4 *out = reinterpret_cast<float4 *>(a.grad[y] + (size_t)e * per) + blockIdx.z * slice;
    if (n == 0) {
        for (size_t i = threadIdx.x; i < slice; i += blockDim.x) out[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        return;
    }
    const float4 *base = reinterpret_cast<const float4 *>(a.scratch + ((size_t)y * a.max_tiles + j) * per) + blockIdx.z * slice;
    for (size_t i = threadIdx.x; i < slice; i += blockDim.x) {
        float4 s = base[i];
        for (int q = 1; q < n; ++q) {
            if (tiles[j + q].rows <= 0) continue;    // balanced tiles: trailing tiles of an expert can be empty
            const float4 v = base[(size_t)q * (per / 4) + i];
            s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
        }
        out[i] = s;
    }
}

template <int R>
static tqp_status launch_projwg_t(tqp_ctx *c, const ProjWgArgs &a, cudaStream_t st) {
    using C = ProjWgCfg<R>;
    if (tqp_status st_attr = ensure_dyn_smem(c, reinterpret_cast<const void *>(&rows_proj_wgrad_kernel<R>), C::SMEM)) return st_attr;
    const Tile *tiles = c->p<Tile>(c->ws.tiles);
    const int32_t *nt = c->p<int32_t>(c->ws.num_tiles);
    rows_proj_wgrad_kernel<R><<<dim3(c->max_tiles, 2), PJ_THREADS, C::SMEM, st>>>(a, tiles, nt);
    TQP_LAUNCH_OK(c);
    projwg_reduce_kernel<<<dim3(c->desc.E, 2, PWR_SPLIT), 256, 0, st>>>(a, tiles, R);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// Z_g = s dG . B_g^T, Z_u = s dU . B_u^T, dB_gate = (s x.A_g)^T dG, dB_up = (s x.A_u)^T dU  (r = 16 / 32; F % 64 == 0).
// map_g / map_u: the tensor maps of dG / dU with box {64, kTileRows}, 128-byte swizzle.
tqp_status launch_rows_proj_wgrad(tqp_ctx *c, const CUtensorMap *map_g, const CUtensorMap *map_u, int F, const bf16 *B_gate, const bf16 *B_up,
                                  const bf16 *XAg, const bf16 *XAu, float s, bf16 *Zg, bf16 *Zu, float *dB_gate, float *dB_up, cudaStream_t st) {
    const int r = c->desc.r;
    ProjWgArgs a;
    a.map[0] = *map_g; a.map[1] = *map_u; a.W[0] = B_gate; a.W[1] = B_up; a.small_[0] = XAg; a.small_[1] = XAu;
    a.out[0] = Zg; a.out[1] = Zu; a.grad[0] = dB_gate; a.grad[1] = dB_up; a.scratch = c->p<float>(c->ws.wg_scratch);
    a.tfirst = c->p<int32_t>(c->ws.tfirst); a.K = F; a.E = c->desc.E; a.max_tiles = c->max_tiles; a.s = s;
    if (r == 16) return launch_projwg_t<16>(c, a, st);
    if (r == 32) return launch_projwg_t<32>(c, a, st);
    return TQP_ERR_ARG;
}

}  // namespace tqp
