// Host-only parts of the path: tridiagonal eigensolve (A8; "the small
// tridiagonal eigenproblem is solved on the host in FP64") and FTLM trace assembly (A9;
// Eqs. 7-9).  No CUDA calls in this file.
#include <algorithm>
#include <cmath>
#include <numeric>
#include <vector>

#include "ftlm_common.cuh"

// Implicit-shift QL iteration on the symmetric tridiagonal (d, e), carrying only the first row z
// of the accumulated rotation product: z_k ends as s_{k,1}, the first component of eigenvector k.
extern "C" int ftlm_tridiag_eig(int m, const double* alpha, const double* beta, double* theta, double* weight) {
  if (m < 0 || (m > 0 && (!alpha || !theta || !weight)) || (m > 1 && !beta)) {
    ftlm_set_error("ftlm_tridiag_eig: bad argument"); return FTLM_EINVAL;
  }
  if (m == 0) return FTLM_OK;
  std::vector<double> d(alpha, alpha + m), e(m, 0.0), z(m, 0.0);
  for (int i = 0; i + 1 < m; ++i) e[i] = beta[i];
  z[0] = 1.0;
  const double eps = 2.220446049250313e-16;
  for (int l = 0; l < m; ++l) {
    int iter = 0;
    int mm;
    do {
      for (mm = l; mm < m - 1; ++mm) {
        const double dd = std::fabs(d[mm]) + std::fabs(d[mm + 1]);
        if (std::fabs(e[mm]) <= eps * dd) break;
      }
      if (mm != l) {
        if (++iter > 200) { ftlm_set_error("ftlm_tridiag_eig: no convergence at l=%d", l); return FTLM_EINVAL; }
        double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
        double r = std::hypot(g, 1.0);
        g = d[mm] - d[l] + e[l] / (g + (g >= 0.0 ? std::fabs(r) : -std::fabs(r)));
        double s = 1.0, c = 1.0, p = 0.0;
        int i;
        for (i = mm - 1; i >= l; --i) {
          double f = s * e[i];
          const double b = c * e[i];
          r = std::hypot(f, g);
          e[i + 1] = r;
          if (r == 0.0) { d[i + 1] -= p; e[mm] = 0.0; break; }
          s = f / r; c = g / r;
          g = d[i + 1] - p;
          r = (d[i] - g) * s + 2.0 * c * b;
          p = s * r;
          d[i + 1] = g + p;
          g = c * r - b;
          f = z[i + 1];
          z[i + 1] = s * z[i] + c * f;
          z[i] = c * z[i] - s * f;
        }
        if (r == 0.0 && i >= l) continue;
        d[l] -= p; e[l] = g; e[mm] = 0.0;
      }
    } while (mm != l);
  }
  std::vector<int> ord(m);
  std::iota(ord.begin(), ord.end(), 0);
  std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return d[a] < d[b]; });
  for (int k = 0; k < m; ++k) { theta[k] = d[ord[k]]; weight[k] = z[ord[k]] * z[ord[k]]; }
  return FTLM_OK;
}

// Eqs. 7-9 with the exponent shift of reading 17.  Moments are accumulated about E_ref
// (variance is shift-invariant), which keeps C = beta^2 (<H^2> - <H>^2) free of cancellation.
extern "C" int ftlm_thermo(int n_sec, const int64_t* dim, const double* Mz, const double* mult, const int* R,
                           int stride, const int* m_eff, const double* theta, const double* weight, int nT,
                           const double* T, double g, double* E_ref, double* Zs, double* E, double* C,
                           double* chi) {
  if (n_sec <= 0 || nT < 0 || !dim || !Mz || !mult || !R || !m_eff || !theta || !weight || (nT > 0 && !T) ||
      !E_ref || stride <= 0) {
    ftlm_set_error("ftlm_thermo: bad argument"); return FTLM_EINVAL;
  }
  double eref = INFINITY;
  int off = 0;
  for (int s = 0; s < n_sec; ++s) {
    if (R[s] <= 0) { ftlm_set_error("ftlm_thermo: sector %d has R <= 0", s); return FTLM_EINVAL; }
    for (int c = 0; c < R[s]; ++c, ++off)
      for (int k = 0; k < m_eff[off]; ++k) eref = std::min(eref, theta[(size_t)off * stride + k]);
  }
  if (!std::isfinite(eref)) { ftlm_set_error("ftlm_thermo: no Ritz values"); return FTLM_EINVAL; }
  *E_ref = eref;
  for (int i = 0; i < nT; ++i) {
    if (!(T[i] > 0.0)) { ftlm_set_error("ftlm_thermo: T[%d] <= 0", i); return FTLM_EINVAL; }
    const double ib = 1.0 / T[i];
    double Z = 0.0, S1 = 0.0, S2 = 0.0, M2 = 0.0;
    off = 0;
    for (int s = 0; s < n_sec; ++s) {
      const double pref = mult[s] * (double)dim[s] / (double)R[s];
      double z = 0.0, s1 = 0.0, s2 = 0.0;
      for (int c = 0; c < R[s]; ++c, ++off) {
        const double* th = theta + (size_t)off * stride;
        const double* w = weight + (size_t)off * stride;
        for (int k = 0; k < m_eff[off]; ++k) {
          const double x = th[k] - eref;
          const double bw = w[k] * std::exp(-x * ib);
          z += bw; s1 += bw * x; s2 += bw * x * x;
        }
      }
      Z += pref * z; S1 += pref * s1; S2 += pref * s2; M2 += Mz[s] * Mz[s] * pref * z;
    }
    const double x1 = S1 / Z, x2 = S2 / Z;
    if (Zs) Zs[i] = Z;
    if (E) E[i] = eref + x1;
    if (C) C[i] = (x2 - x1 * x1) * ib * ib;
    if (chi) chi[i] = g * g * M2 * ib / Z;
  }
  return FTLM_OK;
}
