// TurboQuant-MSE base of the TQP method (PAPER.md L944-948 9.2, L966 9.4, L1047 10.3).
//
//   "the quantizer separates scale from direction, normalizes the vector and stores its norm, applies a seeded random
//    orthogonal rotation, and then quantizes each rotated coordinate independently against a scalar codebook ... the
//    Lloyd-Max scalar codebook for a given dimension and bit width can be computed analytically from that law ... The
//    rotation is a signed Hadamard transform when the dimension is a power of two and a QR rotation from a Gaussian matrix
//    with sign fixing otherwise.  Reconstruction looks up the codebook values and rescales by the stored norm."  (L944-946)
//
// This file holds everything of that format that is not the grouped GEMM itself:
//   tqp_tq_levels      host: Lloyd-Max levels of the coordinate law f_n(y) ~ (1 - y^2)^((n-3)/2)
//   tqp_tq_rotation_qr host: sign-fixed Q of a Gaussian matrix (Gram-Schmidt with re-orthogonalisation)
//   tqp_rotate         activations [rows][n] bf16 -> R x (or R^T y): FWHT kernel / dense bf16 tensor-core product
//   tqp_tq_encode      fp32 rows -> 8-bit codes + fp32 norms (decisions in fp64, as the oracle takes them)
//   tqp_tq_decode      codes + norms -> fp32 rows (reconstruction)
//   tqp_tq_flush       fold s A B into the quantised base in ROTATED space, re-quantise, reset B, telemetry (L966, Table 28)
// Product code: nothing here is shared with oracle/.
#include <cmath>
#include <thread>
#include <vector>

#include "common.cuh"

namespace tqp {

// ======================================================================================================================
// Host: Lloyd-Max levels.  The normalisation of the density cancels in level = int y f / int f, so only
// w(y) = (1 - y^2)^a, a = (n - 3) / 2, is evaluated (as exp(a log1p(-y^2))).  Cells are integrated with a 16-point
// Gauss-Legendre rule on panels no wider than 1/(4 sqrt(n)) (the density's scale is 1/sqrt(n)); beyond 14/sqrt(n) the
// density is below e^-98 of its peak and is dropped.  A few Lloyd sweeps, then Newton's method on the Lloyd-Max equations.
// ======================================================================================================================
namespace {

const double kGLx[8] = {0.0950125098376374, 0.2816035507792589, 0.4580167776572274, 0.6178762444026438,
                        0.7554044083550030, 0.8656312023878318, 0.9445750230732326, 0.9894009349916499};
const double kGLw[8] = {0.1894506104550685, 0.1826034150449236, 0.1691565193950025, 0.1495959888165767,
                        0.1246289712555339, 0.0951585116824928, 0.0622535239386479, 0.0271524594117541};

struct CellInt { double mass, mean; };

CellInt integrate_cell(double lo, double hi, double a, double panel) {
    CellInt r{0.0, 0.0};
    if (hi <= lo) return r;
    const int np = std::max(1, (int)std::ceil((hi - lo) / panel));
    const double h = (hi - lo) / np;
    for (int p = 0; p < np; ++p) {
        const double c = lo + (p + 0.5) * h, hw = 0.5 * h;
        for (int g = 0; g < 8; ++g)
            for (int sgn = -1; sgn <= 1; sgn += 2) {
                const double y = c + sgn * hw * kGLx[g];
                const double w = std::exp(a * std::log1p(-y * y)) * kGLw[g] * hw;
                r.mass += w;
                r.mean += w * y;
            }
    }
    return r;
}

// inverse of the standard normal CDF (bisection on erfc; only used for the starting point)
double inv_norm_cdf(double p) {
    double lo = -12.0, hi = 12.0;
    for (int it = 0; it < 200; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (0.5 * std::erfc(-mid / std::sqrt(2.0)) < p) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

}  // namespace

}  // namespace tqp

extern "C" tqp_status tqp_tq_levels(int n, int bits, double *levels) {
    using namespace tqp;
    if (!levels || n < 8 || bits < 1 || bits > 8) return TQP_ERR_ARG;
    const int L = 1 << bits;
    const double a = 0.5 * (n - 3), sd = 1.0 / std::sqrt((double)n), cut = std::min(1.0, 14.0 * sd), panel = 0.25 * sd;
    std::vector<double> c(L), b(L + 1), cen(L), mass(L);
    for (int j = 0; j < L; ++j) c[j] = std::max(-0.999 * cut, std::min(0.999 * cut, inv_norm_cdf((j + 0.5) / L) * sd));
    auto cells = [&]() {   // boundaries = midpoints; mass and conditional mean of every cell (unnormalised density)
        b[0] = -cut; b[L] = cut;
        for (int j = 1; j < L; ++j) b[j] = 0.5 * (c[j - 1] + c[j]);
        for (int j = 0; j < L; ++j) {
            const CellInt ci = integrate_cell(b[j], b[j + 1], a, panel);
            mass[j] = ci.mass;
            cen[j] = ci.mass > 0 ? ci.mean / ci.mass : c[j];
        }
    };
    for (int it = 0; it < 40; ++it) {   // plain Lloyd sweeps: a robust start (they contract only linearly, far too slowly at 8 bits)
        cells();
        c = cen;
    }
    // Newton on F_j(c) = c_j - E[y | cell_j] = 0; cell j depends on c_{j-1}, c_j, c_{j+1}: tridiagonal Jacobian, Thomas solve
    std::vector<double> dl(L), dg(L), du(L), rhs(L);
    for (int it = 0; it < 100; ++it) {
        cells();
        for (int j = 0; j < L; ++j) {
            const double wlo = j > 0 ? std::exp(a * std::log1p(-b[j] * b[j])) : 0.0;
            const double wup = j < L - 1 ? std::exp(a * std::log1p(-b[j + 1] * b[j + 1])) : 0.0;
            const double dlo = mass[j] > 0 ? -wlo * (b[j] - cen[j]) / mass[j] : 0.0;       // d cen_j / d b_j
            const double dup = mass[j] > 0 ? wup * (b[j + 1] - cen[j]) / mass[j] : 0.0;    // d cen_j / d b_{j+1}
            dg[j] = 1.0 - 0.5 * (dlo + dup);
            dl[j] = -0.5 * dlo;
            du[j] = -0.5 * dup;
            rhs[j] = -(c[j] - cen[j]);
        }
        for (int j = 1; j < L; ++j) {
            const double m = dl[j] / dg[j - 1];
            dg[j] -= m * du[j - 1];
            rhs[j] -= m * rhs[j - 1];
        }
        double step = 0.0;
        rhs[L - 1] /= dg[L - 1];
        for (int j = L - 2; j >= 0; --j) rhs[j] = (rhs[j] - du[j] * rhs[j + 1]) / dg[j];
        for (int j = 0; j < L; ++j) { c[j] += rhs[j]; step = std::max(step, std::fabs(rhs[j])); }
        if (step < 1e-16 * std::max(1.0, 1.0 / sd) * sd * 10.0) break;
    }
    for (int j = 0; j < L / 2; ++j) {   // the law is symmetric: remove the last-bit asymmetry of the solve
        const double v = 0.5 * (c[L - 1 - j] - c[j]);
        c[j] = -v; c[L - 1 - j] = v;
    }
    for (int j = 0; j < L; ++j) levels[j] = c[j];
    return TQP_OK;
}

// Sign-fixed Q of the QR factorisation of a Gaussian matrix G [n][n] (row-major, host): the unique Q with G = Q Rr and
// diag(Rr) > 0 -- what numpy's Householder Q times sign(diag(Rr)) gives.  Classical column Gram-Schmidt done twice
// ("twice is enough"), columns held as contiguous rows of the transposed copy; the updates of the trailing columns
// are spread over host threads.
extern "C" tqp_status tqp_tq_rotation_qr(int n, const double *G, double *R_out) {
    if (!G || !R_out || n < 1) return TQP_ERR_ARG;
    std::vector<double> qt((size_t)n * n);   // qt[j][i] = column j of the working matrix
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) qt[(size_t)j * n + i] = G[(size_t)i * n + j];
    const int nthr = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    for (int k = 0; k < n; ++k) {
        double *qk = &qt[(size_t)k * n];
        double nrm = 0.0;
        for (int i = 0; i < n; ++i) nrm += qk[i] * qk[i];
        nrm = std::sqrt(nrm);
        if (!(nrm > 0.0)) return TQP_ERR_ARG;
        for (int i = 0; i < n; ++i) qk[i] /= nrm;
        auto work = [&](int t) {
            for (int j = k + 1 + t; j < n; j += nthr) {
                double *qj = &qt[(size_t)j * n];
                for (int pass = 0; pass < 2; ++pass) {
                    double dot = 0.0;
                    for (int i = 0; i < n; ++i) dot += qk[i] * qj[i];
                    for (int i = 0; i < n; ++i) qj[i] -= dot * qk[i];
                }
            }
        };
        if (n - k - 1 < 64 || nthr == 1) {
            for (int t = 0; t < nthr; ++t) work(t);
        } else {
            std::vector<std::thread> th;
            for (int t = 0; t < nthr; ++t) th.emplace_back(work, t);
            for (auto &x : th) x.join();
        }
    }
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) R_out[(size_t)i * n + j] = qt[(size_t)j * n + i];
    return TQP_OK;
}

namespace tqp {

// ======================================================================================================================
// Signed Hadamard on rows:  forward  y = H (s . x) / sqrt(n)   (= R x with R = H diag(s) / sqrt(n)),
//                           inverse  x = s . (H y) / sqrt(n)   (= R^T y).
// One CTA per row (grid-stride), the row in shared memory as REAL (float for activations, double for the encoder and
// the flush), log2(n) butterfly stages with one barrier each.  Bound: HBM (2 x rows x n x sizeof(T)); at n = 1024 the
// ten stages of a row take ~1k clk and eight CTAs per SM overlap them.
// ======================================================================================================================
template <typename REAL>
__device__ __forceinline__ void fwht_smem(REAL *v, int n, int tid, int nthr) {
    for (int s = 1; s < n; s <<= 1) {
        __syncthreads();
        for (int b = tid; b < n / 2; b += nthr) {
            const int i = ((b / s) * 2 * s) + (b % s), j = i + s;
            const REAL x = v[i], y = v[j];
            v[i] = x + y;
            v[j] = x - y;
        }
    }
    __syncthreads();
}

// Activation kernel: radix-8 passes.  A row is handled by n / 8 threads; each thread takes its 16-byte chunk of the row
// straight from global memory into registers, does three butterfly stages there, and the later passes (strides 8, 64, 512)
// go registers <-> shared memory with one barrier per pass (4 barriers at n = 1024 instead of 10, two shared-memory
// accesses per element and pass instead of per stage).  Shared rows are padded by one word per 32 (index i -> i + i / 32) so
// that the stride-8 accesses of a pass spread over the banks.  A CTA holds max(1, 1024 / n) rows.  Bound: HBM.
__device__ __forceinline__ int fw_pad(int i) { return i + (i >> 5); }

template <typename T>
__device__ __forceinline__ void fw_load8(const T *p, float (&v)[8]);
template <>
__device__ __forceinline__ void fw_load8<bf16>(const bf16 *p, float (&v)[8]) {
    const uint4 q = *reinterpret_cast<const uint4 *>(p);
    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) { const float2 f = bf16x2_to_float2(w[j]); v[2 * j] = f.x; v[2 * j + 1] = f.y; }
}
template <>
__device__ __forceinline__ void fw_load8<float>(const float *p, float (&v)[8]) {
    const float4 a = *reinterpret_cast<const float4 *>(p), b = *reinterpret_cast<const float4 *>(p + 4);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
template <typename T>
__device__ __forceinline__ void fw_store8(T *p, const float (&v)[8]);
template <>
__device__ __forceinline__ void fw_store8<bf16>(bf16 *p, const float (&v)[8]) {
    uint4 q;
    q.x = float2_to_bf16x2(v[0], v[1]); q.y = float2_to_bf16x2(v[2], v[3]); q.z = float2_to_bf16x2(v[4], v[5]); q.w = float2_to_bf16x2(v[6], v[7]);
    *reinterpret_cast<uint4 *>(p) = q;
}
template <>
__device__ __forceinline__ void fw_store8<float>(float *p, const float (&v)[8]) {
    *reinterpret_cast<float4 *>(p) = make_float4(v[0], v[1], v[2], v[3]);
    *reinterpret_cast<float4 *>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
}
// butterflies over the low `nb` bits of the register index
__device__ __forceinline__ void fw_bfly8(float (&v)[8], int nb) {
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        if (b < nb) {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                if (!(k & (1 << b))) { const float x = v[k], y = v[k | (1 << b)]; v[k] = x + y; v[k | (1 << b)] = x - y; }
        }
    }
}

// MODE 0: Y = rotation of X.  MODE 1 (bf16): Y = R (silu(X) * X2) -- the SwiGLU of the TurboQuant layer with the rotation of its
// result in the same pass (h is never rounded or stored unrotated).  MODE 2 (bf16, inverse): dh = R^T X, then the SwiGLU
// backward against the saved g = X2, u = X3:  Y = dg, Y2 = du  (dh stays in registers).
template <typename TIN, typename TOUT, int MODE>
__global__ void __launch_bounds__(1024) tq_fwht_rows_kernel(const TIN *__restrict__ X, TOUT *__restrict__ Y, long long rows, int n, int logn,
                                                             const int8_t *__restrict__ signs, int inverse, const TIN *__restrict__ X2,
                                                             const TIN *__restrict__ X3, TOUT *__restrict__ Y2) {
    extern __shared__ float fw_s[];
    const int tpr = n / 8, rpc = blockDim.x / tpr;             // threads per row, rows per CTA
    const int lr = threadIdx.x / tpr, t = threadIdx.x % tpr, lane = threadIdx.x % 32;
    float *sm = fw_s + lr * fw_pad(n);
    const float rs = rsqrtf((float)n);
    float sg[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) sg[k] = (float)signs[8 * t + k];
    // bits 3 .. 7 of the element index are lane bits (a row's threads are consecutive lanes): butterflies by shuffle
    const int nsh = min(logn, 8) - 3;
    float fl[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) fl[b] = (lane >> b) & 1 ? -1.f : 1.f;
    // shared-memory passes for bits 8 and up (n > 256): element slots of this thread per pass, fixed for the whole kernel
    int idx[2][8];
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        const int ls = 8 + 3 * p, nb = max(0, min(3, logn - ls)), s = 1 << ls;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int kb = k & ((1 << nb) - 1), rem = t * (8 >> nb) + (k >> nb);
            idx[p][k] = fw_pad(((rem >> ls) << (ls + nb)) | (kb << ls) | (rem & (s - 1)));
        }
    }
    for (long long row0 = (long long)blockIdx.x * rpc; row0 < rows; row0 += (long long)gridDim.x * rpc) {
        const long long row = row0 + lr;
        const bool act = row < rows;
        float v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = 0.f;
        if (act) {
            fw_load8<TIN>(X + row * n + 8 * t, v);
            if (MODE == 1) {
                float u[8];
                fw_load8<TIN>(X2 + row * n + 8 * t, u);
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = v[k] / (1.f + __expf(-v[k])) * u[k];
            }
            if (!inverse) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] *= sg[k];
            }
        }
        fw_bfly8(v, 3);                                          // bits 0..2
#pragma unroll
        for (int b = 0; b < 5; ++b) {                            // bits 3..7: v = partner + (upper lane ? -v : v)
            if (b < nsh) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = fmaf(v[k], fl[b], __shfl_xor_sync(0xffffffffu, v[k], 1 << b));
            }
        }
        if (logn > 8) {
#pragma unroll
            for (int k = 0; k < 8; ++k) sm[fw_pad(8 * t + k)] = v[k];
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                const int ls = 8 + 3 * p;
                if (ls < logn) {
                    __syncthreads();
#pragma unroll
                    for (int k = 0; k < 8; ++k) v[k] = sm[idx[p][k]];
                    fw_bfly8(v, min(3, logn - ls));
#pragma unroll
                    for (int k = 0; k < 8; ++k) sm[idx[p][k]] = v[k];
                }
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = sm[fw_pad(8 * t + k)];
            __syncthreads();
        }
        if (act) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                v[k] *= rs;
                if (inverse) v[k] *= sg[k];
            }
            if (MODE == 2) {   // v = dh: sig = sigmoid(g); du = dh g sig; dg = dh u sig (1 + g (1 - sig))
                float g[8], u[8], dg[8];
                fw_load8<TIN>(X2 + row * n + 8 * t, g);
                fw_load8<TIN>(X3 + row * n + 8 * t, u);
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const float sig = 1.f / (1.f + __expf(-g[k]));
                    dg[k] = v[k] * u[k] * sig * (1.f + g[k] * (1.f - sig));
                    v[k] = v[k] * g[k] * sig;
                }
                fw_store8<TOUT>(Y + row * n + 8 * t, dg);
                fw_store8<TOUT>(Y2 + row * n + 8 * t, v);
            } else {
                fw_store8<TOUT>(Y + row * n + 8 * t, v);
            }
        }
    }
}

// Adapter tensors between [E][L][r] (dir 0 in) and [E][r][L] (dir 1 in), r <= 32 the adapter rank, L the layer width: a CTA takes
// 256 positions of L, reads its 256 r elements as one contiguous run and writes r runs of 256 (or the reverse).
template <typename T>
__global__ void __launch_bounds__(256) tq_transpose_kernel(const T *__restrict__ in, T *__restrict__ out, int L, int r, int dir) {
    __shared__ T tile[32][257];
    const size_t e = blockIdx.y;
    const int l0 = blockIdx.x * 256, nl = min(256, L - l0);
    const T *src = in + e * (size_t)L * r;
    T *dst = out + e * (size_t)L * r;
    if (dir == 0) {
        for (int v = threadIdx.x; v < nl * r; v += 256) tile[v % r][v / r] = src[(size_t)l0 * r + v];
        __syncthreads();
        for (int q = 0; q < r; ++q)
            for (int l = threadIdx.x; l < nl; l += 256) dst[(size_t)q * L + l0 + l] = tile[q][l];
    } else {
        for (int q = 0; q < r; ++q)
            for (int l = threadIdx.x; l < nl; l += 256) tile[q][l] = src[(size_t)q * L + l0 + l];
        __syncthreads();
        for (int v = threadIdx.x; v < nl * r; v += 256) dst[(size_t)l0 * r + v] = tile[v % r][v / r];
    }
}

// ======================================================================================================================
// Dense rotation of activations:  C[rows][n] = X[rows][n] . Rm^T  with Rm [n][n] bf16 row-major (both operands K-major).
// Forward: Rm = R (y = R x); inverse: Rm = R^T.  Plain tensor-core product (mma.sync m16n8k16, bf16 in, fp32 accumulate):
// CTA tile 128 x 128 x 32, 8 warps of 64 x 32, 3-stage cp.async ring, ldmatrix from rows padded to 40 elements.
// SPLIT: the input is fp32 and goes in as hi + lo bf16 parts (two MMAs per k-step) -- used for the adapter gradients,
// where one more bf16 rounding of the data would cost accuracy.
// ======================================================================================================================
constexpr int DR_BM = 128, DR_BN = 128, DR_BK = 32, DR_LD = 40, DR_ST = 3;

__device__ __forceinline__ void dr_ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void dr_mma(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void dr_cp16(uint32_t dst, const void *src, bool ok) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(ok ? 16 : 0) : "memory");
}

template <bool SPLIT, typename TOUT>
__global__ void __launch_bounds__(256) tq_dense_rot_kernel(const void *__restrict__ Xv, const bf16 *__restrict__ Rm, TOUT *__restrict__ C,
                                                           long long rows, int n) {
    extern __shared__ __align__(16) uint8_t dr_raw[];
    constexpr int A_PARTS = SPLIT ? 2 : 1;
    bf16 *as = reinterpret_cast<bf16 *>(dr_raw);                                   // [ST][A_PARTS][BM][LD]
    bf16 *bs = as + (size_t)DR_ST * A_PARTS * DR_BM * DR_LD;                        // [ST][BN][LD]
    const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
    const long long m0 = (long long)blockIdx.y * DR_BM;
    const int n0 = blockIdx.x * DR_BN;
    const int wm = (warp / 4) * 64, wn = (warp % 4) * 32;
    float acc[4][4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[i][j][q] = 0.f;
    const int nk = n / DR_BK;
    auto load = [&](int kt, int st) {
        const int k0 = kt * DR_BK;
        // B tile: 128 rows x 32 k = 512 chunks of 8 bf16
        for (int v = tid; v < DR_BN * (DR_BK / 8); v += 256) {
            const int r = v / (DR_BK / 8), c8 = (v % (DR_BK / 8)) * 8;
            dr_cp16((uint32_t)__cvta_generic_to_shared(bs + ((size_t)st * DR_BN + r) * DR_LD + c8), Rm + (size_t)(n0 + r) * n + k0 + c8, true);
        }
        if (!SPLIT) {
            const bf16 *X = reinterpret_cast<const bf16 *>(Xv);
            for (int v = tid; v < DR_BM * (DR_BK / 8); v += 256) {
                const int r = v / (DR_BK / 8), c8 = (v % (DR_BK / 8)) * 8;
                const bool ok = m0 + r < rows;
                dr_cp16((uint32_t)__cvta_generic_to_shared(as + ((size_t)st * DR_BM + r) * DR_LD + c8), X + (size_t)(ok ? m0 + r : 0) * n + k0 + c8, ok);
            }
        } else {   // fp32 source: registers -> hi / lo bf16 parts
            const float *X = reinterpret_cast<const float *>(Xv);
            for (int v = tid; v < DR_BM * (DR_BK / 4); v += 256) {
                const int r = v / (DR_BK / 4), c4 = (v % (DR_BK / 4)) * 4;
                float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
                if (m0 + r < rows) f = *reinterpret_cast<const float4 *>(X + (size_t)(m0 + r) * n + k0 + c4);
                const float fv[4] = {f.x, f.y, f.z, f.w};
                bf16 *hi = as + (((size_t)st * 2 + 0) * DR_BM + r) * DR_LD + c4, *lo = as + (((size_t)st * 2 + 1) * DR_BM + r) * DR_LD + c4;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const bf16 h = __float2bfloat16_rn(fv[q]);
                    hi[q] = h;
                    lo[q] = __float2bfloat16_rn(fv[q] - __bfloat162float(h));
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    for (int s = 0; s < DR_ST - 1; ++s) {
        if (s < nk) load(s, s); else asm volatile("cp.async.commit_group;" ::: "memory");
    }
    for (int kt = 0; kt < nk; ++kt) {
        asm volatile("cp.async.wait_group %0;" ::"n"(DR_ST - 2) : "memory");
        __syncthreads();
        if (kt + DR_ST - 1 < nk) load(kt + DR_ST - 1, (kt + DR_ST - 1) % DR_ST); else asm volatile("cp.async.commit_group;" ::: "memory");
        const int st = kt % DR_ST;
#pragma unroll
        for (int ks = 0; ks < DR_BK / 16; ++ks) {
            uint32_t bfr[2][4];   // two n16 blocks: regs {n0-7 k0-7, n0-7 k8-15, n8-15 k0-7, n8-15 k8-15}
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int r = wn + j * 16 + (lane % 8) + 8 * (lane / 16), c = ks * 16 + 8 * ((lane / 8) % 2);
                dr_ldsm_x4((uint32_t)__cvta_generic_to_shared(bs + ((size_t)st * DR_BN + r) * DR_LD + c), bfr[j]);
            }
#pragma unroll
            for (int part = 0; part < A_PARTS; ++part)
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    uint32_t af[4];   // m16 x k16: regs {m0-7 k0-7, m8-15 k0-7, m0-7 k8-15, m8-15 k8-15}
                    const int r = wm + i * 16 + (lane % 16), c = ks * 16 + 8 * (lane / 16);
                    dr_ldsm_x4((uint32_t)__cvta_generic_to_shared(as + (((size_t)st * A_PARTS + part) * DR_BM + r) * DR_LD + c), af);
#pragma unroll
                    for (int j = 0; j < 4; ++j) dr_mma(acc[i][j], af, bfr[j / 2][(j % 2) * 2], bfr[j / 2][(j % 2) * 2 + 1]);
                }
        }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    const int g = lane / 4, t = lane % 4;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const long long row = m0 + wm + i * 16 + g + 8 * h;
            if (row >= rows) continue;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int col = n0 + wn + j * 8 + 2 * t;
                const float v0 = acc[i][j][2 * h], v1 = acc[i][j][2 * h + 1];
                if (sizeof(TOUT) == 2) *reinterpret_cast<uint32_t *>(C + (size_t)row * n + col) = float2_to_bf16x2(v0, v1);
                else *reinterpret_cast<float2 *>(C + (size_t)row * n + col) = make_float2(v0, v1);
            }
        }
}

// R (fp64, row-major) -> bf16 R, bf16 R^T and fp64 R^T (one-time, per rotation)
__global__ void tq_prepare_dense_kernel(const double *__restrict__ R, int n, bf16 *__restrict__ Rb, bf16 *__restrict__ Rtb, double *__restrict__ Rt) {
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)n * n) return;
    const int i = (int)(idx / n), j = (int)(idx % n);
    const double v = R[idx];
    Rb[idx] = __float2bfloat16_rn((float)v);
    Rtb[(size_t)j * n + i] = __float2bfloat16_rn((float)v);
    Rt[(size_t)j * n + i] = v;
}

}  // namespace tqp

namespace tqp {

// ======================================================================================================================
// Encoder / decoder / flush.  All decisions that end in an integer code are taken in fp64, the precision the oracle
// (numpy) takes them in; a code can then differ from the oracle's only where a rotated coordinate lies within a few ulp
// of a cell boundary.  One CTA per weight row; the row lives in shared memory as doubles.
// ======================================================================================================================
__device__ __forceinline__ double block_sum(double v, double *red) {   // fixed order: lanes by xor-tree, warps in sequence
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    __syncthreads();
    if (threadIdx.x % 32 == 0) red[threadIdx.x / 32] = v;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < (int)(blockDim.x / 32); ++w) s += red[w];
    return s;
}

// searchsorted(bounds, y, side = "left"): the number of boundaries strictly below y; a coordinate ON a boundary takes the lower code
__device__ __forceinline__ int tq_code_of(const double *bounds, int nb, double y) {
    int lo = 0, hi = nb;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (bounds[mid] < y) lo = mid + 1; else hi = mid;
    }
    return lo;
}

struct TqRowArgs {
    int n, hadamard;
    const int8_t *signs;      // [n]
    const double *R, *Rt;     // dense: R[j][i], Rt[i][j]
    const double *levels;     // [256]
};

// y = R u for the row in v[] (dense: result written to y[], a second smem array; Hadamard: in place, y == v)
__device__ __forceinline__ void tq_rotate_row(const TqRowArgs &a, double *v, double *y) {
    const int n = a.n;
    if (a.hadamard) {
        for (int i = threadIdx.x; i < n; i += blockDim.x) v[i] *= (double)a.signs[i];
        fwht_smem(v, n, threadIdx.x, blockDim.x);
        const double rs = 1.0 / sqrt((double)n);
        for (int i = threadIdx.x; i < n; i += blockDim.x) v[i] *= rs;
        __syncthreads();
    } else {
        __syncthreads();
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            double acc = 0.0;
            for (int i = 0; i < n; ++i) acc += a.Rt[(size_t)i * n + j] * v[i];
            y[j] = acc;
        }
        __syncthreads();
    }
}

// mode 0: encode fp32 rows W.  mode 1: flush -- the row is formed in rotated space from the stored base and the rotated
// adapter:  v[i] = norm * levels[code[i]] + s * sum_q Arot[e][i][q] * B[e][q][o]   (fold the delta in).
struct TqEncArgs {
    TqRowArgs rot;
    const float *W;              // mode 0: [rows][n]
    uint8_t *codes;              // [rows][n]   (mode 1: read, then overwritten)
    float *norms;                // [rows]
    const double *Arot;          // mode 1: [E][n][r] fp64 = R . A[e]
    const bf16 *B;               // mode 1: [E][r][out]
    int r, out_dim;              // rows = E * out_dim
    double s;
    double *tele;                // mode 1: [rows][2] = (|base row|^2, |delta row|^2)
};

template <int MODE>
__global__ void __launch_bounds__(256) tq_encode_kernel(const TqEncArgs a, long long rows) {
    extern __shared__ double enc_s[];
    const int n = a.rot.n;
    double *v = enc_s, *y = a.rot.hadamard ? enc_s : enc_s + n, *bounds = enc_s + (a.rot.hadamard ? n : 2 * n), *red = bounds + 256;
    for (int j = threadIdx.x; j < 255; j += blockDim.x) bounds[j] = 0.5 * (a.rot.levels[j] + a.rot.levels[j + 1]);
    for (long long row = blockIdx.x; row < rows; row += gridDim.x) {
        __syncthreads();
        double ss = 0.0, sb = 0.0, sd = 0.0;
        if (MODE == 0) {
            const float *w = a.W + row * n;
            for (int i = threadIdx.x; i < n; i += blockDim.x) {
                const double x = (double)w[i];
                v[i] = x;
                ss += x * x;
            }
        } else {
            const long long e = row / a.out_dim;
            const int o = (int)(row % a.out_dim);
            const uint8_t *cr = a.codes + row * n;
            const double nrm = (double)a.norms[row];
            const double *ar = a.Arot + (size_t)e * n * a.r;
            const bf16 *bc = a.B + (size_t)e * a.r * a.out_dim + o;
            double bq[32];
            for (int q = 0; q < a.r; ++q) bq[q] = (double)__bfloat162float(bc[(size_t)q * a.out_dim]);
            for (int i = threadIdx.x; i < n; i += blockDim.x) {
                double dl = 0.0;
                for (int q = 0; q < a.r; ++q) dl += ar[(size_t)i * a.r + q] * bq[q];
                dl *= a.s;
                const double base = nrm * a.rot.levels[cr[i]];
                const double x = base + dl;
                v[i] = x;
                ss += x * x; sb += base * base; sd += dl * dl;
            }
        }
        const double tot = block_sum(ss, red);
        if (MODE == 1) {
            const double tb = block_sum(sb, red), td = block_sum(sd, red);
            if (threadIdx.x == 0) { a.tele[2 * row] = tb; a.tele[2 * row + 1] = td; }
        }
        const double nrm = sqrt(tot);
        if (threadIdx.x == 0) a.norms[row] = (float)nrm;
        const double inv = nrm > 0.0 ? 1.0 / nrm : 0.0;
        __syncthreads();
        // u = row / norm: the oracle divides (np.divide), so divide here too (x * (1 / norm) rounds differently)
        for (int i = threadIdx.x; i < n; i += blockDim.x) v[i] = nrm > 0.0 ? v[i] / nrm : 0.0;
        (void)inv;
        if (MODE == 1) {
            // the row already is R W_merged: no rotation
            __syncthreads();
            uint8_t *cw = a.codes + row * n;
            for (int i = threadIdx.x; i < n; i += blockDim.x) cw[i] = (uint8_t)tq_code_of(bounds, 255, v[i]);
        } else {
            __syncthreads();
            tq_rotate_row(a.rot, v, y);
            uint8_t *cw = a.codes + row * n;
            for (int i = threadIdx.x; i < n; i += blockDim.x) cw[i] = (uint8_t)tq_code_of(bounds, 255, y[i]);
        }
    }
}

// Reconstruction (L946): W[row][:] = norm * (levels[codes] R)
__global__ void __launch_bounds__(256) tq_decode_kernel(const TqRowArgs rot, const uint8_t *__restrict__ codes, const float *__restrict__ norms,
                                                        long long rows, float *__restrict__ W) {
    extern __shared__ double enc_s[];
    const int n = rot.n;
    double *v = enc_s;
    for (long long row = blockIdx.x; row < rows; row += gridDim.x) {
        __syncthreads();
        const uint8_t *cr = codes + row * n;
        for (int i = threadIdx.x; i < n; i += blockDim.x) v[i] = rot.levels[cr[i]];
        const double nrm = (double)norms[row];
        float *w = W + row * n;
        if (rot.hadamard) {   // x = s . H yh / sqrt(n)
            fwht_smem(v, n, threadIdx.x, blockDim.x);
            const double rs = 1.0 / sqrt((double)n);
            for (int i = threadIdx.x; i < n; i += blockDim.x) w[i] = (float)(v[i] * rs * (double)rot.signs[i] * nrm);
        } else {
            __syncthreads();
            for (int i = threadIdx.x; i < n; i += blockDim.x) {
                double acc = 0.0;
                for (int j = 0; j < n; ++j) acc += v[j] * rot.R[(size_t)j * n + i];
                w[i] = (float)(acc * nrm);
            }
        }
    }
}

// Arot[e][j][q] = sum_i R[j][i] A[e][i][q]  (fp64).  Hadamard: one CTA per (e, q), the column in shared memory.
__global__ void __launch_bounds__(256) tq_rotate_adapter_had_kernel(const TqRowArgs rot, const bf16 *__restrict__ A, int r, double *__restrict__ Arot) {
    extern __shared__ double enc_s[];
    const int n = rot.n, e = blockIdx.x / r, q = blockIdx.x % r;
    const bf16 *src = A + (size_t)e * n * r + q;
    for (int i = threadIdx.x; i < n; i += blockDim.x) enc_s[i] = (double)__bfloat162float(src[(size_t)i * r]) * (double)rot.signs[i];
    fwht_smem(enc_s, n, threadIdx.x, blockDim.x);
    const double rs = 1.0 / sqrt((double)n);
    double *dst = Arot + (size_t)e * n * r + q;
    for (int i = threadIdx.x; i < n; i += blockDim.x) dst[(size_t)i * r] = enc_s[i] * rs;
}
// dense: grid (ceil(n / 256), E), thread j
__global__ void __launch_bounds__(256) tq_rotate_adapter_dense_kernel(const TqRowArgs rot, const bf16 *__restrict__ A, int r, double *__restrict__ Arot) {
    const int n = rot.n, e = blockIdx.y, j = blockIdx.x * 256 + threadIdx.x;
    if (j >= n) return;
    double acc[32];
    for (int q = 0; q < 32; ++q) acc[q] = 0.0;
    const bf16 *src = A + (size_t)e * n * r;
    for (int i = 0; i < n; ++i) {
        const double rji = rot.Rt[(size_t)i * n + j];
        for (int q = 0; q < r; ++q) acc[q] += rji * (double)__bfloat162float(src[(size_t)i * r + q]);
    }
    for (int q = 0; q < r; ++q) Arot[((size_t)e * n + j) * r + q] = acc[q];
}

// Table 28 telemetry per expert: tele_out[e] = (|s A B|_F, |W| / (|W| + |s A B|)) from the per-row partial sums, in row order
__global__ void tq_flush_telemetry_kernel(const double *__restrict__ tele, int out_dim, float *__restrict__ out) {
    const int e = blockIdx.x;
    if (threadIdx.x != 0) return;
    double sb = 0.0, sd = 0.0;
    for (int o = 0; o < out_dim; ++o) { sb += tele[2 * ((size_t)e * out_dim + o)]; sd += tele[2 * ((size_t)e * out_dim + o) + 1]; }
    const double nb = sqrt(sb), na = sqrt(sd);
    out[2 * e] = (float)na;
    out[2 * e + 1] = (float)(nb + na > 0.0 ? nb / (nb + na) : 1.0);
}

}  // namespace tqp

// ======================================================================================================================
// Host side
// ======================================================================================================================
namespace tqp {

#define TQ_REQ(ctx, cond, code, msg) do { if (!(cond)) { (ctx)->err = msg; return code; } } while (0)

static bool pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

tqp_status tq_check_space(tqp_ctx *c, const tqp_tq_space *sp) {
    TQ_REQ(c, sp != nullptr, TQP_ERR_ARG, "tqp_tq_space is NULL");
    TQ_REQ(c, sp->n >= 64 && sp->n <= 8192 && sp->n % 64 == 0, TQP_ERR_SHAPE, "tqp_tq_space.n must be a multiple of 64 in [64, 8192]");
    TQ_REQ(c, sp->levels != nullptr, TQP_ERR_ARG, "tqp_tq_space.levels is NULL");
    if (sp->hadamard) {
        TQ_REQ(c, pow2(sp->n), TQP_ERR_SHAPE, "signed Hadamard needs a power-of-two width (PAPER.md L946)");
        TQ_REQ(c, sp->signs != nullptr, TQP_ERR_ARG, "tqp_tq_space.signs is NULL");
    } else {
        TQ_REQ(c, sp->R != nullptr, TQP_ERR_ARG, "tqp_tq_space.R is NULL");
    }
    return TQP_OK;
}

// derived copies of a dense rotation (bf16 R and R^T for the activation product, fp64 R^T for coalesced fp64 reads);
// library-owned device memory, built on first use, freed by tqp_destroy
tqp_status tq_dense_rot(tqp_ctx *c, const tqp_tq_space *sp, cudaStream_t st, const TqRot **out) {
    for (const TqRot &r : c->tq_rots)
        if (r.R == sp->R && r.n == sp->n) { *out = &r; return TQP_OK; }
    TqRot r{};
    r.R = sp->R; r.n = sp->n;
    const size_t nn = (size_t)sp->n * sp->n;
    TQP_CUDA_OK(c, cudaMalloc(&r.Rb, nn * 2));
    TQP_CUDA_OK(c, cudaMalloc(&r.Rtb, nn * 2));
    TQP_CUDA_OK(c, cudaMalloc(&r.Rt, nn * 8));
    tq_prepare_dense_kernel<<<(unsigned)((nn + 255) / 256), 256, 0, st>>>(sp->R, sp->n, r.Rb, r.Rtb, r.Rt);
    TQP_LAUNCH_OK(c);
    c->tq_rots.push_back(r);
    *out = &c->tq_rots.back();
    return TQP_OK;
}

tqp_status tq_row_args(tqp_ctx *c, const tqp_tq_space *sp, cudaStream_t st, TqRowArgs *a) {
    a->n = sp->n; a->hadamard = sp->hadamard; a->signs = sp->signs; a->R = sp->R; a->Rt = nullptr; a->levels = sp->levels;
    if (!sp->hadamard) {
        const TqRot *r;
        if (tqp_status s = tq_dense_rot(c, sp, st, &r)) return s;
        a->Rt = r->Rt;
    }
    return TQP_OK;
}

// rows [rows][n] of bf16 (or fp32 when in_f32) -> rotated rows, bf16 (or fp32 when out_f32)
tqp_status launch_tq_rotate(tqp_ctx *c, const tqp_tq_space *sp, const void *X, bool in_f32, long long rows, void *Y, bool out_f32, int inverse,
                            cudaStream_t st) {
    if (rows <= 0) return TQP_OK;
    const int n = sp->n;
    if (sp->hadamard) {
        const int tpr = n / 8, rpc = std::max(1, 128 / tpr), thr = tpr * rpc;   // >= 128 threads per CTA, whole rows
        int logn = 0;
        while ((1 << logn) < n) ++logn;
        const long long ctas = (rows + rpc - 1) / rpc;
        const int grid = (int)std::min<long long>(ctas, (long long)c->num_sms * std::max(1, 2048 / thr));
        const size_t sm = (size_t)rpc * (n + n / 32) * 4;
        if (in_f32 && out_f32) tq_fwht_rows_kernel<float, float, 0><<<grid, thr, sm, st>>>((const float *)X, (float *)Y, rows, n, logn, sp->signs, inverse, nullptr, nullptr, nullptr);
        else if (in_f32) tq_fwht_rows_kernel<float, bf16, 0><<<grid, thr, sm, st>>>((const float *)X, (bf16 *)Y, rows, n, logn, sp->signs, inverse, nullptr, nullptr, nullptr);
        else if (out_f32) tq_fwht_rows_kernel<bf16, float, 0><<<grid, thr, sm, st>>>((const bf16 *)X, (float *)Y, rows, n, logn, sp->signs, inverse, nullptr, nullptr, nullptr);
        else tq_fwht_rows_kernel<bf16, bf16, 0><<<grid, thr, sm, st>>>((const bf16 *)X, (bf16 *)Y, rows, n, logn, sp->signs, inverse, nullptr, nullptr, nullptr);
        TQP_LAUNCH_OK(c);
        return TQP_OK;
    }
    TQ_REQ(c, n % DR_BN == 0, TQP_ERR_SHAPE, "dense rotation needs n % 128 == 0");
    const TqRot *r;
    if (tqp_status s = tq_dense_rot(c, sp, st, &r)) return s;
    const bf16 *Rm = inverse ? r->Rtb : r->Rb;
    dim3 grid(n / DR_BN, (unsigned)((rows + DR_BM - 1) / DR_BM));
    const int parts = in_f32 ? 2 : 1;
    const int sm = DR_ST * (parts * DR_BM + DR_BN) * DR_LD * 2;
    if (in_f32) {
        TQ_REQ(c, out_f32, TQP_ERR_ARG, "fp32 rows rotate to fp32 rows");
        if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_dense_rot_kernel<true, float>), sm)) return s;
        tq_dense_rot_kernel<true, float><<<grid, 256, sm, st>>>(X, Rm, (float *)Y, rows, n);
    } else if (out_f32) {
        if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_dense_rot_kernel<false, float>), sm)) return s;
        tq_dense_rot_kernel<false, float><<<grid, 256, sm, st>>>(X, Rm, (float *)Y, rows, n);
    } else {
        if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_dense_rot_kernel<false, bf16>), sm)) return s;
        tq_dense_rot_kernel<false, bf16><<<grid, 256, sm, st>>>(X, Rm, (bf16 *)Y, rows, n);
    }
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

__global__ void tq_make_lut_kernel(const double *__restrict__ levels, bf16 *__restrict__ lut) {
    lut[threadIdx.x] = __float2bfloat16_rn((float)levels[threadIdx.x]);
}
tqp_status launch_tq_make_lut(tqp_ctx *c, const double *levels, bf16 *lut, cudaStream_t st) {
    tq_make_lut_kernel<<<1, 256, 0, st>>>(levels, lut);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// Hadamard spaces only: H' = R (silu(G) * U)   /   dG, dU from dH' = R dh and the saved G, U   (one pass each)
tqp_status launch_tq_swiglu_fwd_rot(tqp_ctx *c, const tqp_tq_space *sp, const bf16 *G, const bf16 *U, bf16 *Hr, long long rows, cudaStream_t st) {
    const int n = sp->n, tpr = n / 8, rpc = std::max(1, 128 / tpr), thr = tpr * rpc;
    int logn = 0;
    while ((1 << logn) < n) ++logn;
    const int grid = (int)std::min<long long>((rows + rpc - 1) / rpc, (long long)c->num_sms * std::max(1, 2048 / thr));
    tq_fwht_rows_kernel<bf16, bf16, 1><<<grid, thr, (size_t)rpc * (n + n / 32) * 4, st>>>(G, Hr, rows, n, logn, sp->signs, 0, U, nullptr, nullptr);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
tqp_status launch_tq_swiglu_bwd_rot(tqp_ctx *c, const tqp_tq_space *sp, const bf16 *dHr, const bf16 *G, const bf16 *U, bf16 *dG, bf16 *dU,
                                    long long rows, cudaStream_t st) {
    const int n = sp->n, tpr = n / 8, rpc = std::max(1, 128 / tpr), thr = tpr * rpc;
    int logn = 0;
    while ((1 << logn) < n) ++logn;
    const int grid = (int)std::min<long long>((rows + rpc - 1) / rpc, (long long)c->num_sms * std::max(1, 2048 / thr));
    tq_fwht_rows_kernel<bf16, bf16, 2><<<grid, thr, (size_t)rpc * (n + n / 32) * 4, st>>>(dHr, dG, rows, n, logn, sp->signs, 1, G, U, dU);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

// ---- rotation of the adapters along their STRIDED dimension: A[e][i][q] (i < n, q < r): FWHT over i for every (e, q) --------
// (replaces transpose -> row FWHT -> transpose for Hadamard spaces: three passes over the tensor and two temporaries become
// one pass.)  CTA = (expert, group of 8 columns).  The rows come in coalesced (8 values = 16 / 32 bytes of every row), are
// spread into 8 column vectors in shared memory (fp32, padded like the row kernel's), every column goes through the row
// kernel's passes (registers for bits 0-2 of the index, shuffles for bits 3-7, shared memory above), and the rows go out
// coalesced again.  Forward: y = H (signs * x) / sqrt(n); inverse: x = signs * (H y) / sqrt(n).
// CG values of one row: 8 / 16 bytes (bf16) or 16 / 32 bytes (fp32)
template <typename T, int CG>
__device__ __forceinline__ void fs_load(const T *p, float (&v)[CG]) {
    if constexpr (sizeof(T) == 2) {
        uint32_t w[CG / 2];
        if constexpr (CG == 8) { const uint4 q = *reinterpret_cast<const uint4 *>(p); w[0] = q.x; w[1] = q.y; w[2] = q.z; w[3] = q.w; }
        else { const uint2 q = *reinterpret_cast<const uint2 *>(p); w[0] = q.x; w[1] = q.y; }
#pragma unroll
        for (int j = 0; j < CG / 2; ++j) { const float2 f = bf16x2_to_float2(w[j]); v[2 * j] = f.x; v[2 * j + 1] = f.y; }
    } else {
#pragma unroll
        for (int j = 0; j < CG / 4; ++j) {
            const float4 q = *reinterpret_cast<const float4 *>(p + 4 * j);
            v[4 * j] = q.x; v[4 * j + 1] = q.y; v[4 * j + 2] = q.z; v[4 * j + 3] = q.w;
        }
    }
}
template <typename T, int CG>
__device__ __forceinline__ void fs_store(T *p, const float (&v)[CG]) {
    if constexpr (sizeof(T) == 2) {
        uint32_t w[CG / 2];
#pragma unroll
        for (int j = 0; j < CG / 2; ++j) w[j] = float2_to_bf16x2(v[2 * j], v[2 * j + 1]);
        if constexpr (CG == 8) *reinterpret_cast<uint4 *>(p) = make_uint4(w[0], w[1], w[2], w[3]);
        else *reinterpret_cast<uint2 *>(p) = make_uint2(w[0], w[1]);
    } else {
#pragma unroll
        for (int j = 0; j < CG / 4; ++j) *reinterpret_cast<float4 *>(p + 4 * j) = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
    }
}

template <typename T, int CG>
__global__ void __launch_bounds__(1024) tq_fwht_strided_kernel(const T *__restrict__ X, T *__restrict__ Y, int n, int logn, int r,
                                                                const int8_t *__restrict__ signs, int inverse) {
    extern __shared__ float fs_s[];
    const int np = n + n / 32;   // floats per column
    const T *src = X + (size_t)blockIdx.y * n * r + blockIdx.x * CG;
    T *dst = Y + (size_t)blockIdx.y * n * r + blockIdx.x * CG;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        float v[CG];
        fs_load<T, CG>(src + (size_t)i * r, v);
        const float sg = inverse ? 1.f : (float)signs[i];
#pragma unroll
        for (int c = 0; c < CG; ++c) fs_s[c * np + fw_pad(i)] = v[c] * sg;
    }
    __syncthreads();
    const int tpr = n / 8, cpi = blockDim.x / tpr;             // threads per column, columns per round (blockDim = tpr * cpi, cpi | CG)
    const int lr = threadIdx.x / tpr, t = threadIdx.x % tpr, lane = threadIdx.x % 32;
    const float rs = rsqrtf((float)n);
    const int nsh = min(logn, 8) - 3;
    float fl[5];
#pragma unroll
    for (int b = 0; b < 5; ++b) fl[b] = (lane >> b) & 1 ? -1.f : 1.f;
    int idx[2][8];
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        const int ls = 8 + 3 * p, nb = max(0, min(3, logn - ls)), s = 1 << ls;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int kb = k & ((1 << nb) - 1), rem = t * (8 >> nb) + (k >> nb);
            idx[p][k] = fw_pad(((rem >> ls) << (ls + nb)) | (kb << ls) | (rem & (s - 1)));
        }
    }
    float sgo[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) sgo[k] = inverse ? (float)signs[8 * t + k] : 1.f;
    for (int cb = 0; cb < CG; cb += cpi) {
        float *sm = fs_s + (cb + lr) * np;
        float v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = sm[fw_pad(8 * t + k)];
        fw_bfly8(v, 3);
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            if (b < nsh) {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = fmaf(v[k], fl[b], __shfl_xor_sync(0xffffffffu, v[k], 1 << b));
            }
        }
        if (logn > 8) {
#pragma unroll
            for (int k = 0; k < 8; ++k) sm[fw_pad(8 * t + k)] = v[k];
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                const int ls = 8 + 3 * p;
                if (ls < logn) {
                    __syncthreads();
#pragma unroll
                    for (int k = 0; k < 8; ++k) v[k] = sm[idx[p][k]];
                    fw_bfly8(v, min(3, logn - ls));
#pragma unroll
                    for (int k = 0; k < 8; ++k) sm[idx[p][k]] = v[k];
                }
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = sm[fw_pad(8 * t + k)];
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) sm[fw_pad(8 * t + k)] = v[k] * rs * sgo[k];
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        float v[CG];
#pragma unroll
        for (int c = 0; c < CG; ++c) v[c] = fs_s[c * np + fw_pad(i)];
        fs_store<T, CG>(dst + (size_t)i * r, v);
    }
}

// Y[e][i][q] = rotation along i of X[e][i][q]  (Hadamard spaces, 128 <= n <= 8192, r % 8 == 0); X may equal Y
template <typename T>
tqp_status launch_tq_fwht_strided(tqp_ctx *c, const tqp_tq_space *sp, const T *X, T *Y, int E, int r, int inverse, cudaStream_t st) {
    const int n = sp->n;
    TQ_REQ(c, sp->hadamard && n >= 128 && n <= 8192 && r % 8 == 0, TQP_ERR_ARG, "strided FWHT: Hadamard space, 128 <= n <= 8192, r % 8 == 0");
    int logn = 0;
    while ((1 << logn) < n) ++logn;
    // eight columns per CTA (135 KB of shared memory at n = 4096, one CTA per SM): 78 / 96 us per bf16 / fp32 adapter pack at
    // cfg 5; four columns and two CTAs per SM were slower (fp32: 106 us)
    constexpr int CG = 8;
    const int tpr = n / 8, cpi = std::max(1, std::min(CG, 1024 / tpr));
    const int smem = CG * (n + n / 32) * 4;
    if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_fwht_strided_kernel<T, CG>), smem)) return s;
    tq_fwht_strided_kernel<T, CG><<<dim3(r / CG, E), tpr * cpi, smem, st>>>(X, Y, n, logn, r, sp->signs, inverse);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
template tqp_status launch_tq_fwht_strided<bf16>(tqp_ctx *, const tqp_tq_space *, const bf16 *, bf16 *, int, int, int, cudaStream_t);
template tqp_status launch_tq_fwht_strided<float>(tqp_ctx *, const tqp_tq_space *, const float *, float *, int, int, int, cudaStream_t);

template <typename T>
tqp_status launch_tq_transpose(tqp_ctx *c, const T *in, T *out, int E, int a, int b, cudaStream_t st) {
    // [E][a][b] -> [E][b][a]; one of a, b is the rank
    const int dir = b <= 32 ? 0 : 1, L = dir == 0 ? a : b, r = dir == 0 ? b : a;
    if (r > 32) { c->err = "transpose: neither side is an adapter rank"; return TQP_ERR_ARG; }
    dim3 grid((L + 255) / 256, E);
    tq_transpose_kernel<T><<<grid, 256, 0, st>>>(in, out, L, r, dir);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}
template tqp_status launch_tq_transpose<bf16>(tqp_ctx *, const bf16 *, bf16 *, int, int, int, cudaStream_t);
template tqp_status launch_tq_transpose<float>(tqp_ctx *, const float *, float *, int, int, int, cudaStream_t);

static size_t enc_smem(const tqp_tq_space *sp) { return ((size_t)(sp->hadamard ? 1 : 2) * sp->n + 256 + 32) * 8; }

}  // namespace tqp

using namespace tqp;

extern "C" {

tqp_status tqp_rotate(tqp_ctx *c, const tqp_tq_space *sp, const void *X, long long rows, void *Y, int inverse, void *stream) {
    if (!c) return TQP_ERR_ARG;
    c->launches = 0;
    if (tqp_status s = tq_check_space(c, sp)) return s;
    TQ_REQ(c, X && Y && rows >= 0, TQP_ERR_ARG, "NULL tensor or negative rows");
    return launch_tq_rotate(c, sp, X, false, rows, Y, false, inverse ? 1 : 0, (cudaStream_t)stream);
}

tqp_status tqp_tq_encode(tqp_ctx *c, const tqp_tq_space *sp, const float *W, long long rows, uint8_t *codes, float *norms, void *stream) {
    if (!c) return TQP_ERR_ARG;
    c->launches = 0;
    if (tqp_status s = tq_check_space(c, sp)) return s;
    TQ_REQ(c, W && codes && norms && rows >= 0, TQP_ERR_ARG, "NULL tensor or negative rows");
    if (rows == 0) return TQP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    TqEncArgs a{};
    if (tqp_status s = tq_row_args(c, sp, st, &a.rot)) return s;
    a.W = W; a.codes = codes; a.norms = norms;
    const size_t sm = enc_smem(sp);
    if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_encode_kernel<0>), (int)sm)) return s;
    tq_encode_kernel<0><<<(int)std::min<long long>(rows, (long long)c->num_sms * 4), 256, sm, st>>>(a, rows);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

tqp_status tqp_tq_decode(tqp_ctx *c, const tqp_tq_space *sp, const uint8_t *codes, const float *norms, long long rows, float *W, void *stream) {
    if (!c) return TQP_ERR_ARG;
    c->launches = 0;
    if (tqp_status s = tq_check_space(c, sp)) return s;
    TQ_REQ(c, W && codes && norms && rows >= 0, TQP_ERR_ARG, "NULL tensor or negative rows");
    if (rows == 0) return TQP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    TqRowArgs ra;
    if (tqp_status s = tq_row_args(c, sp, st, &ra)) return s;
    const size_t sm = (size_t)sp->n * 8;
    if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_decode_kernel), (int)sm)) return s;
    tq_decode_kernel<<<(int)std::min<long long>(rows, (long long)c->num_sms * 4), 256, sm, st>>>(ra, codes, norms, rows, W);
    TQP_LAUNCH_OK(c);
    return TQP_OK;
}

tqp_status tqp_tq_flush(tqp_ctx *c, const tqp_tq_space *sp, int n_experts, int out_dim, int r, float lora_scale, uint8_t *codes, float *norms,
                        void *A, void *B, const void *A_new, float *telemetry, void *stream) {
    if (!c) return TQP_ERR_ARG;
    c->launches = 0;
    if (tqp_status s = tq_check_space(c, sp)) return s;
    TQ_REQ(c, codes && norms && A && B, TQP_ERR_ARG, "NULL tensor");
    TQ_REQ(c, n_experts >= 0 && out_dim > 0 && r >= 1 && r <= 32, TQP_ERR_ARG, "n_experts >= 0, out_dim > 0, 1 <= r <= 32");
    if (n_experts == 0) return TQP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const int n = sp->n;
    const long long rows = (long long)n_experts * out_dim;
    TqEncArgs a{};
    if (tqp_status s = tq_row_args(c, sp, st, &a.rot)) return s;
    double *Arot = nullptr, *tele = nullptr;
    TQP_CUDA_OK(c, cudaMallocAsync(&Arot, (size_t)n_experts * n * r * 8, st));
    TQP_CUDA_OK(c, cudaMallocAsync(&tele, (size_t)rows * 2 * 8, st));
    if (sp->hadamard) {
        const size_t sm = (size_t)n * 8;
        if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_rotate_adapter_had_kernel), (int)sm)) return s;
        tq_rotate_adapter_had_kernel<<<n_experts * r, 256, sm, st>>>(a.rot, (const bf16 *)A, r, Arot);
    } else {
        tq_rotate_adapter_dense_kernel<<<dim3((n + 255) / 256, n_experts), 256, 0, st>>>(a.rot, (const bf16 *)A, r, Arot);
    }
    TQP_LAUNCH_OK(c);
    a.codes = codes; a.norms = norms; a.Arot = Arot; a.B = (const bf16 *)B; a.r = r; a.out_dim = out_dim; a.s = (double)lora_scale; a.tele = tele;
    TqEncArgs af = a;
    af.rot.hadamard = 1;   // the flush row is already in rotated space: the kernel needs one row buffer only
    const size_t sm = ((size_t)n + 256 + 32) * 8;
    if (tqp_status s = ensure_dyn_smem(c, reinterpret_cast<const void *>(&tq_encode_kernel<1>), (int)sm)) return s;
    tq_encode_kernel<1><<<(int)std::min<long long>(rows, (long long)c->num_sms * 4), 256, sm, st>>>(af, rows);
    TQP_LAUNCH_OK(c);
    if (telemetry) {
        tq_flush_telemetry_kernel<<<n_experts, 32, 0, st>>>(tele, out_dim, telemetry);
        TQP_LAUNCH_OK(c);
    }
    // reset the adapter factors (L966): B <- 0, A <- the caller's fresh draw if given
    TQP_CUDA_OK(c, cudaMemsetAsync(B, 0, (size_t)n_experts * r * out_dim * 2, st));
    if (A_new) TQP_CUDA_OK(c, cudaMemcpyAsync(A, A_new, (size_t)n_experts * n * r * 2, cudaMemcpyDeviceToDevice, st));
    TQP_CUDA_OK(c, cudaFreeAsync(Arot, st));
    TQP_CUDA_OK(c, cudaFreeAsync(tele, st));
    return TQP_OK;
}

}  // extern "C"
