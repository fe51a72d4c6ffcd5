/* CPU ORACLE, C / OpenMP twin -- test infrastructure, NOT a product path.
 *
 * The same plain definitions as oracle/oracle_np.py (which stays the reference the pins of
 * tests/test_oracle_*.py are written against), restated as row loops in C so that the large
 * BASELINE.json configurations (1.5e9 stored entries) can be checked in full and so that the
 * CPU baseline bench.py reports runs on all host cores (SURVEY.md 8(d) "Oracle timing").
 * Nothing here is blocked, fused or reordered beyond "rows are dealt to threads and every
 * thread keeps its own per-gene accumulators, added up at the end"; float64 / int64 throughout.
 * It shares no code with paper_2603_02402_b200/csrc and is pinned element-wise against
 * oracle_np in tests/test_oracle_c.py (integers equal, floats within 1e-12).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.  Citations are PAPER.md lines.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC oracle_c.c -o liboracle_c.so -lm   (oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void orc_set_num_threads(int t) {
#ifdef _OPENMP
  if (t > 0) omp_set_num_threads(t);
#else
  (void)t;
#endif
}

/* Q1..Q4 ("QC metrics", cell-wise on CSR; readings R1..R4 of DESIGN.md):
 *   T_i = sum (int64) x, N_i = #{x != 0}, M_i = sum over flagged genes, pct_i = 100 M_i / T_i,
 *   C_j = #{x != 0 in column j}, T_j = sum (int64) x in column j.
 * gene_n_cells / gene_total are ADDED to (the caller zeroes them; row chunks accumulate). */
void orc_qc(int64_t n, int32_t G, const int64_t* indptr, const int32_t* indices, const float* data,
            const uint8_t* flags, int64_t* cell_total, int32_t* cell_n_genes, int64_t* cell_flag_total,
            float* cell_pct, int64_t* gene_n_cells, int64_t* gene_total) {
#pragma omp parallel
  {
    int64_t* cnt = (int64_t*)calloc((size_t)G, sizeof(int64_t));
    int64_t* tot = (int64_t*)calloc((size_t)G, sizeof(int64_t));
#pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
      int64_t T = 0, M = 0;
      int32_t N = 0;
      for (int64_t p = indptr[i]; p < indptr[i + 1]; ++p) {
        const float x = data[p];
        const int64_t xi = (int64_t)(double)x; /* truncation */
        const int32_t j = indices[p];
        T += xi;
        if (x != 0.0f) { ++N; ++cnt[j]; }
        if (flags != NULL && flags[j] != 0) M += xi;
        tot[j] += xi;
      }
      cell_total[i] = T;
      cell_n_genes[i] = N;
      cell_flag_total[i] = M;
      cell_pct[i] = (float)(100.0 * (double)M / (double)T); /* 0/0 -> NaN (R3) */
    }
#pragma omp critical
    {
      for (int32_t j = 0; j < G; ++j) { gene_n_cells[j] += cnt[j]; gene_total[j] += tot[j]; }
    }
    free(cnt);
    free(tot);
  }
}

/* N1 + L1: x' = (float)((double) x * (s / T_i)), one rounding (R5); a cell with
 * T_i == 0 is left untouched (R3); x'' = (float) log1p((double) x').  Either output may be NULL. */
void orc_normalize_log1p(int64_t n, const int64_t* indptr, const float* data, const int64_t* cell_total,
                         double target_sum, float* x_norm, float* x_log) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < n; ++i) {
    const double T = (double)cell_total[i];
    const double scale = T != 0.0 ? target_sum / T : 1.0;
    for (int64_t p = indptr[i]; p < indptr[i + 1]; ++p) {
      const float xn = (float)((double)data[p] * scale);
      if (x_norm != NULL) x_norm[p] = xn;
      if (x_log != NULL) x_log[p] = (float)log1p((double)xn);
    }
  }
}

/* M1, sums ("per-gene mean and variance", L137): S1_j += sum v, S2_j += sum v^2,
 * stored_j += number of stored entries, v = x (transform 0) or expm1(x) (transform 1, R8).
 * ADDED to the outputs (row chunks accumulate). */
void orc_gene_sums(int64_t n, int32_t G, const int64_t* indptr, const int32_t* indices, const float* data,
                   int transform, double* S1, double* S2, double* stored) {
#pragma omp parallel
  {
    double* a1 = (double*)calloc((size_t)G, sizeof(double));
    double* a2 = (double*)calloc((size_t)G, sizeof(double));
    double* ac = (double*)calloc((size_t)G, sizeof(double));
#pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
      for (int64_t p = indptr[i]; p < indptr[i + 1]; ++p) {
        double v = (double)data[p];
        if (transform == 1) v = expm1(v);
        const int32_t j = indices[p];
        a1[j] += v;
        a2[j] += v * v;
        ac[j] += 1.0;
      }
    }
#pragma omp critical
    {
      for (int32_t j = 0; j < G; ++j) { S1[j] += a1[j]; S2[j] += a2[j]; stored[j] += ac[j]; }
    }
    free(a1);
    free(a2);
    free(ac);
  }
}

/* M1, second pass of the textbook two-pass variance: SS_j += sum over stored entries of
 * (v - mean_j)^2; the caller adds (n - stored_j) mean_j^2 and divides by (n - ddof). */
void orc_gene_sqdev(int64_t n, int32_t G, const int64_t* indptr, const int32_t* indices, const float* data,
                    int transform, const double* mean, double* SS) {
#pragma omp parallel
  {
    double* a = (double*)calloc((size_t)G, sizeof(double));
#pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
      for (int64_t p = indptr[i]; p < indptr[i + 1]; ++p) {
        double v = (double)data[p];
        if (transform == 1) v = expm1(v);
        const int32_t j = indices[p];
        const double d = v - mean[j];
        a[j] += d * d;
      }
    }
#pragma omp critical
    {
      for (int32_t j = 0; j < G; ++j) SS[j] += a[j];
    }
    free(a);
  }
}
