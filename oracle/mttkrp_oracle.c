/*
 * fp64 CPU oracle for all-mode sparse MTTKRP.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or helper with the
 * CUDA path under paper_2405_08470_b200/csrc/ and is never a fallback for it.
 *
 * What it computes is the plain definition the paper's method reaches exactly (up to
 * rounding order):
 *   PAPER.md:121 (Sec. 2.1.5, elementwise computation)
 *       C(i2,r) = C(i2,r) + val(X(i0,i1,i2)) . A(i0,r) o B(i1,r)
 *   PAPER.md:100 (Eq. 1)   A~ = X_(0)(B (.) C), ...  generalised to N modes:
 *       Y_d[i_d, r] = sum over nonzeros k of val_k * prod_{m != d} A_m[i_m(k), r]
 *   PAPER.md:206-216 (Alg. 2): l(r) <- value; for each input mode w != d: l(r) <- l(r) * vec(r);
 *       Y_d(c_d, r) <- Y_d(c_d, r) + l(r)
 * in double precision, visiting the nonzeros in the mode-d order (PAPER.md:145, :177:
 * the tensor is ordered by the output mode), which is a stable sort of the COO list.
 *
 * DESIGN.md readings used here: output is overwritten, rows without nonzeros are 0
 * (reading 2); duplicate coordinates add (reading 10); indices are 0-based (reading 11);
 * inputs are fp32 and are widened to fp64 before any arithmetic (reading 12).
 *
 * Pins (tests/test_oracle_pins.py): dense unfold x explicit Khatri-Rao brute force, the
 * all-ones closed form, the cross-mode invariant, scipy.sparse SpMM for N=2, bincount for
 * R=1, linearity / permutation / duplicate-splitting properties, numpy lexsort for the
 * permutation.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/*
 * Stable sort of the nonzeros by the key tuple (i_{order[0]}, i_{order[1]}, ...), ties keeping
 * the original COO order: perm[k] = original position of the element at sorted position k.
 * Implemented as LSD passes of a stable counting sort, least significant key first
 * ("order the hyperedges ... assign a remap id reflecting its position";
 * PAPER.md:299 Observation 1: the remap id is unique per element, i.e. perm is a bijection).
 * idx is SoA: idx[m*nnz + k].  Returns 0, or -1 on allocation failure / bad index.
 */
int oracle_sort_perm(int nmodes, const int64_t *dims, int64_t nnz, const int32_t *idx,
                     int nkeys, const int32_t *order, int64_t *perm)
{
    int64_t *cur = perm;
    int64_t *tmp = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nnz > 0 ? nnz : 1));
    if (!tmp) return -1;
    for (int64_t k = 0; k < nnz; ++k) cur[k] = k;
    for (int p = nkeys - 1; p >= 0; --p) {
        int m = order[p];
        if (m < 0 || m >= nmodes) { free(tmp); return -1; }
        int64_t size = dims[m];
        int64_t *count = (int64_t *)calloc((size_t)size + 1, sizeof(int64_t));
        if (!count) { free(tmp); return -1; }
        const int32_t *key = idx + (size_t)m * (size_t)nnz;
        for (int64_t k = 0; k < nnz; ++k) {
            int32_t v = key[k];
            if (v < 0 || v >= size) { free(count); free(tmp); return -1; }
            count[v + 1]++;
        }
        for (int64_t v = 0; v < size; ++v) count[v + 1] += count[v];
        for (int64_t k = 0; k < nnz; ++k) {          /* forward scan keeps ties in order */
            int64_t src = cur[k];
            tmp[count[key[src]]++] = src;
        }
        memcpy(cur, tmp, sizeof(int64_t) * (size_t)nnz);
        free(count);
    }
    free(tmp);
    return 0;
}

/*
 * Y_d (I_d x R, fp64, row-major) and the error normaliser
 *   S_d[i,r] = sum_k |val_k| * prod_{m != d} |A_m[i_m(k), r]|
 * visiting nonzeros in the order perm[0..nnz) (perm == NULL: COO order).
 * factors[m] is I_m x R row-major fp32; factors[d] is not read.
 * Y and S are fully overwritten.  S may be NULL.
 */
int oracle_mttkrp_mode(int nmodes, const int64_t *dims, int64_t nnz, const int32_t *idx,
                       const float *vals, const float *const *factors, int R, int d,
                       const int64_t *perm, double *Y, double *S)
{
    if (d < 0 || d >= nmodes || R <= 0) return -1;
    size_t out = (size_t)dims[d] * (size_t)R;
    memset(Y, 0, sizeof(double) * out);
    if (S) memset(S, 0, sizeof(double) * out);
    double *l = (double *)malloc(sizeof(double) * (size_t)R * 2);
    if (!l) return -1;
    double *labs = l + R;
    for (int64_t p = 0; p < nnz; ++p) {
        int64_t k = perm ? perm[p] : p;
        double v = (double)vals[k];
        for (int r = 0; r < R; ++r) { l[r] = v; labs[r] = fabs(v); }   /* Alg. 2 line 8 */
        for (int w = 0; w < nmodes; ++w) {                             /* Alg. 2 line 9 */
            if (w == d) continue;
            int64_t c = idx[(size_t)w * (size_t)nnz + (size_t)k];
            const float *vec = factors[w] + (size_t)c * (size_t)R;     /* Alg. 2 line 10 */
            for (int r = 0; r < R; ++r) {                              /* Alg. 2 lines 12-13 */
                double a = (double)vec[r];
                l[r] *= a;
                labs[r] *= fabs(a);
            }
        }
        int64_t cd = idx[(size_t)d * (size_t)nnz + (size_t)k];
        double *y = Y + (size_t)cd * (size_t)R;
        for (int r = 0; r < R; ++r) y[r] += l[r];                      /* Alg. 2 lines 14-15 */
        if (S) {
            double *s = S + (size_t)cd * (size_t)R;
            for (int r = 0; r < R; ++r) s[r] += labs[r];
        }
    }
    free(l);
    return 0;
}

/*
 * Row-partitioned multi-core variant used only for timing the CPU baseline: perm must be a
 * mode-d order (keys non-decreasing), rows are split across threads and every row is summed
 * by one thread in perm order, so the result is bit-identical to oracle_mttkrp_mode for any
 * thread count.  Returns the number of threads used, or -1.
 */
int oracle_mttkrp_mode_rows(int nmodes, const int64_t *dims, int64_t nnz, const int32_t *idx,
                            const float *vals, const float *const *factors, int R, int d,
                            const int64_t *perm, double *Y, double *S, int nthreads)
{
    if (d < 0 || d >= nmodes || R <= 0 || !perm) return -1;
    int64_t rows = dims[d];
    size_t out = (size_t)rows * (size_t)R;
    memset(Y, 0, sizeof(double) * out);
    if (S) memset(S, 0, sizeof(double) * out);
    /* row_start[i] = first sorted position of row i */
    int64_t *row_start = (int64_t *)calloc((size_t)rows + 1, sizeof(int64_t));
    if (!row_start) return -1;
    const int32_t *kd = idx + (size_t)d * (size_t)nnz;
    for (int64_t p = 0; p < nnz; ++p) row_start[kd[perm[p]] + 1]++;
    for (int64_t i = 0; i < rows; ++i) row_start[i + 1] += row_start[i];
    for (int64_t p = 1; p < nnz; ++p)
        if (kd[perm[p - 1]] > kd[perm[p]]) { free(row_start); return -1; }
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
#endif
        double *l = (double *)malloc(sizeof(double) * (size_t)R * 2);
        double *labs = l + R;
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 64)
#endif
        for (int64_t i = 0; i < rows; ++i) {
            double *y = Y + (size_t)i * (size_t)R;
            double *s = S ? S + (size_t)i * (size_t)R : NULL;
            for (int64_t p = row_start[i]; p < row_start[i + 1]; ++p) {
                int64_t k = perm[p];
                double v = (double)vals[k];
                for (int r = 0; r < R; ++r) { l[r] = v; labs[r] = fabs(v); }
                for (int w = 0; w < nmodes; ++w) {
                    if (w == d) continue;
                    int64_t c = idx[(size_t)w * (size_t)nnz + (size_t)k];
                    const float *vec = factors[w] + (size_t)c * (size_t)R;
                    for (int r = 0; r < R; ++r) {
                        double a = (double)vec[r];
                        l[r] *= a;
                        labs[r] *= fabs(a);
                    }
                }
                for (int r = 0; r < R; ++r) y[r] += l[r];
                if (s) for (int r = 0; r < R; ++r) s[r] += labs[r];
            }
        }
        free(l);
#ifdef _OPENMP
    }
#endif
    free(row_start);
    return used;
}

/* Selected output rows only (full-size sampled parity): rows[j] -> Ysel[j,:], Ssel[j,:].
 * One pass over the nonzeros in COO order restricted to the wanted rows, in the order
 * perm gives (perm == NULL: COO order). */
int oracle_mttkrp_rows_subset(int nmodes, const int64_t *dims, int64_t nnz, const int32_t *idx,
                              const float *vals, const float *const *factors, int R, int d,
                              const int64_t *perm, int64_t nsel, const int64_t *rows,
                              double *Ysel, double *Ssel)
{
    if (d < 0 || d >= nmodes || R <= 0) return -1;
    int64_t nrows = dims[d];
    int64_t *slot = (int64_t *)malloc(sizeof(int64_t) * (size_t)nrows);
    if (!slot) return -1;
    for (int64_t i = 0; i < nrows; ++i) slot[i] = -1;
    for (int64_t j = 0; j < nsel; ++j) {
        if (rows[j] < 0 || rows[j] >= nrows) { free(slot); return -1; }
        slot[rows[j]] = j;
    }
    memset(Ysel, 0, sizeof(double) * (size_t)nsel * (size_t)R);
    if (Ssel) memset(Ssel, 0, sizeof(double) * (size_t)nsel * (size_t)R);
    double *l = (double *)malloc(sizeof(double) * (size_t)R * 2);
    double *labs = l + R;
    const int32_t *kd = idx + (size_t)d * (size_t)nnz;
    for (int64_t p = 0; p < nnz; ++p) {
        int64_t k = perm ? perm[p] : p;
        int64_t j = slot[kd[k]];
        if (j < 0) continue;
        double v = (double)vals[k];
        for (int r = 0; r < R; ++r) { l[r] = v; labs[r] = fabs(v); }
        for (int w = 0; w < nmodes; ++w) {
            if (w == d) continue;
            int64_t c = idx[(size_t)w * (size_t)nnz + (size_t)k];
            const float *vec = factors[w] + (size_t)c * (size_t)R;
            for (int r = 0; r < R; ++r) {
                double a = (double)vec[r];
                l[r] *= a;
                labs[r] *= fabs(a);
            }
        }
        double *y = Ysel + (size_t)j * (size_t)R;
        for (int r = 0; r < R; ++r) y[r] += l[r];
        if (Ssel) {
            double *s = Ssel + (size_t)j * (size_t)R;
            for (int r = 0; r < R; ++r) s[r] += labs[r];
        }
    }
    free(l);
    free(slot);
    return 0;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
