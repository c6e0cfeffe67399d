/* FP64 CPU oracle, large-N part (plain C + OpenMP).  TEST INFRASTRUCTURE ONLY.
 *
 * Same plain definitions as oracle/ftlm_oracle.py (which pins this file on small cases):
 * explicit enumeration of the sector basis, binary search in the sorted basis
 * as the state-to-index map (L119), the row-wise gather of Eq. 12 (L105-L109) at s = 1/2 in
 * float64, and the Lanczos recursion of L45 (reading 7 of DESIGN.md).  Shares no code, header
 * or table with the CUDA library.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC ftlm_oracle_c.c -o libftlm_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Explicit enumeration: every label in [0, 2^N) is visited and kept iff its popcount is N_up.
 * The label space is cut into equal chunks only so that threads can count, then fill, in
 * ascending order.  basis == NULL: count only.  Returns the sector dimension. */
int64_t orc_enumerate(int N, int N_up, uint64_t *basis) {
  const uint64_t total = 1ull << N;
  const int nchunk = 1024;
  const uint64_t step = (total + nchunk - 1) / nchunk;
  int64_t *cnt = (int64_t *)calloc(nchunk + 1, sizeof(int64_t));
#pragma omp parallel for schedule(dynamic, 4)
  for (int c = 0; c < nchunk; ++c) {
    uint64_t lo = (uint64_t)c * step, hi = lo + step;
    if (hi > total) hi = total;
    int64_t k = 0;
    for (uint64_t n = lo; n < hi; ++n) k += (__builtin_popcountll(n) == N_up);
    cnt[c + 1] = k;
  }
  for (int c = 0; c < nchunk; ++c) cnt[c + 1] += cnt[c];
  int64_t D = cnt[nchunk];
  if (basis) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int c = 0; c < nchunk; ++c) {
      uint64_t lo = (uint64_t)c * step, hi = lo + step;
      if (hi > total) hi = total;
      int64_t k = cnt[c];
      for (uint64_t n = lo; n < hi; ++n)
        if (__builtin_popcountll(n) == N_up) basis[k++] = n;
    }
  }
  free(cnt);
  return D;
}

/* Binary search in the ascending basis; -1 if absent (Alg. 2 step 2 convention). */
int64_t orc_index(const uint64_t *basis, int64_t D, uint64_t label) {
  int64_t lo = 0, hi = D - 1;
  while (lo <= hi) {
    int64_t mid = lo + ((hi - lo) >> 1);
    uint64_t b = basis[mid];
    if (b == label) return mid;
    if (b < label) lo = mid + 1; else hi = mid - 1;
  }
  return -1;
}

void orc_index_many(const uint64_t *basis, int64_t D, const uint64_t *labels, int64_t n,
                    int64_t *out) {
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < n; ++k) out[k] = orc_index(basis, D, labels[k]);
}

/* y[row] for row in [row0, row0 + nrows): Eq. 12 at s = 1/2.
 * diag = sum_b J_b m_i m_j - h M_z; off-diagonal J_b/2 on antiparallel bonds. */
void orc_apply_rows(int N, int nb, const int32_t *bi, const int32_t *bj, const double *J,
                    double h, int N_up, const uint64_t *basis, int64_t D, const double *v,
                    int64_t row0, int64_t nrows, double *y) {
  const double zee = -h * ((double)N_up - 0.5 * (double)N);
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < nrows; ++r) {
    const int64_t t = row0 + r;
    const uint64_t n = basis[t];
    double diag = zee, acc = 0.0;
    for (int b = 0; b < nb; ++b) {
      const int si = (int)((n >> bi[b]) & 1u), sj = (int)((n >> bj[b]) & 1u);
      if (si == sj) {
        diag += 0.25 * J[b];
      } else {
        diag -= 0.25 * J[b];
        const uint64_t src = n ^ (1ull << bi[b]) ^ (1ull << bj[b]);
        acc += 0.5 * J[b] * v[orc_index(basis, D, src)];
      }
    }
    y[r] = diag * v[t] + acc;
  }
}

/* Same row loop, but v is not stored: element u of the input is produced by the caller's
 * table `vs` over a sparse set; used for sampled rows at N = 34 where only the needed
 * entries are generated.  src_idx[r*nb + b] receives the source index (or -1). */
void orc_neighbors_rows(int N, int nb, const int32_t *bi, const int32_t *bj,
                        const uint64_t *basis, int64_t D, const int64_t *rows, int64_t nrows,
                        int64_t *src_idx) {
  (void)N;
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < nrows; ++r) {
    const uint64_t n = basis[rows[r]];
    for (int b = 0; b < nb; ++b) {
      const int si = (int)((n >> bi[b]) & 1u), sj = (int)((n >> bj[b]) & 1u);
      src_idx[r * nb + b] =
          (si == sj) ? -1 : orc_index(basis, D, n ^ (1ull << bi[b]) ^ (1ull << bj[b]));
    }
  }
}

static double dot(const double *a, const double *b, int64_t n) {
  double s = 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
  for (int64_t k = 0; k < n; ++k) s += a[k] * b[k];
  return s;
}

/* Lanczos of L45 / reading 7; q1 is consumed as q_1.  Returns m_eff; alpha[m_eff],
 * beta[m_eff-1].  Breakdown: beta_j <= tol * max_k(|alpha_k|, beta_k) (reading 10). */
int orc_lanczos(int N, int nb, const int32_t *bi, const int32_t *bj, const double *J, double h,
                int N_up, const uint64_t *basis, int64_t D, const double *q1, int n_steps,
                double tol, double *alpha, double *beta) {
  int m = n_steps < D ? n_steps : (int)D;
  double *q = (double *)malloc(sizeof(double) * D);
  double *qp = (double *)calloc(D, sizeof(double));
  double *w = (double *)malloc(sizeof(double) * D);
  memcpy(q, q1, sizeof(double) * D);
  double beta_prev = 0.0, scale = 0.0;
  int m_eff = 0;
  for (int j = 1; j <= m; ++j) {
    orc_apply_rows(N, nb, bi, bj, J, h, N_up, basis, D, q, 0, D, w);
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < D; ++k) w[k] -= beta_prev * qp[k];
    const double a = dot(q, w, D);
    alpha[j - 1] = a;
    m_eff = j;
    if (j == m) break;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < D; ++k) w[k] -= a * q[k];
    const double bn = sqrt(dot(w, w, D));
    if (fabs(a) > scale) scale = fabs(a);
    if (bn > scale) scale = bn;
    if (bn <= tol * scale) break;
    beta[j - 1] = bn;
    double *tmp = qp; qp = q; q = tmp;          /* q_prev <- q_j */
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < D; ++k) q[k] = w[k] / bn;
    beta_prev = bn;
  }
  free(q); free(qp); free(w);
  return m_eff;
}
