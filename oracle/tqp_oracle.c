/* ======================================================================================================
 * TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH.
 *
 * CPU oracle of the routed-expert layer of the TQP method ("Reversible Foundations", arxiv 2606.07404):
 * top-k router -> permutation by expert -> grouped SwiGLU FFN over vector-quantised frozen weights plus
 * rank-r adapters (forward and backward) -> weighted combine.  Written from PAPER.md (§3.4, Table 4
 * L237-239, §5.1, §9.1, §9.2, §10.6) and, where the paper fixes no format,
 * from the readings listed in DESIGN.md ("Readings of the paper", R1-R20).  Plain loops, no blocking, no
 * BLAS; fp32 (the precision BASELINE.json north_star names) and fp64 instantiations of the same text.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this
 * library.  It shares no code with paper_2606_07404_b200/csrc and neither side imports the other.
 *
 * Pins (tests/test_oracle_pins.py): P1 closed-form dequant, P2 B=0 adapters, P3 brute-force top-k with
 * injected ties, P4 permutation invariants, P5 fp64 finite differences, P6 softmax special cases,
 * P7 E=1 dense FFN vs an independent numpy fp64 matmul, P8 merge identity, P9 linearity /
 * empty experts, P10 fp32-vs-fp64, P12 hand-checkable 0/1 worked example (tests/golden/p12_worked_example.txt),
 * P13 hand-computed combine / combine_bwd with k = 3 and distinct rows (tests/golden/p13_combine_worked_example.txt);
 * P5 also runs at lora_scale 0.5 and 2 with large adapters (the factor s in dA, dB and the adapter term of dX).
 * Parity unpinned: absolute numerical outputs — the paper prints no worked example, codebook or expected
 * value for this layer.
 * ====================================================================================================== */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define CAT_(a, b) a##b
#define CAT(a, b) CAT_(a, b)

#define REAL float
#define FN(name) CAT(name, _f32)
#define FMA fmaf
#define EXP expf
#include "tqp_oracle_impl.inc"
#undef REAL
#undef FN
#undef FMA
#undef EXP

#define REAL double
#define FN(name) CAT(name, _f64)
#define FMA fma
#define EXP exp
#include "tqp_oracle_impl.inc"
#undef REAL
#undef FN
#undef FMA
#undef EXP

/* Step 5, "expert dispatch" (Table 6): stable counting sort of the flat assignment
 * index a = t*k+j by expert id.  counts[e] = #{a: idx[a]=e}; offsets = exclusive scan (offsets[E] = N);
 * within an expert rows are in ascending a; perm[p] = a, inv_perm[a] = p.  Integer-only. */
void tqp_oracle_dispatch(const int32_t *topk_idx, int T, int k, int E,
                         int32_t *counts, int32_t *offsets, int32_t *perm, int32_t *inv_perm)
{
    int N = T * k;
    for (int e = 0; e < E; ++e) counts[e] = 0;
    for (int a = 0; a < N; ++a) counts[topk_idx[a]] += 1;
    offsets[0] = 0;
    for (int e = 0; e < E; ++e) offsets[e + 1] = offsets[e] + counts[e];
    int32_t *cursor = (int32_t *)malloc((size_t)E * sizeof(int32_t));
    for (int e = 0; e < E; ++e) cursor[e] = offsets[e];
    for (int a = 0; a < N; ++a) {
        int p = cursor[topk_idx[a]]++;
        perm[p] = a;
        inv_perm[a] = p;
    }
    free(cursor);
}

int tqp_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
