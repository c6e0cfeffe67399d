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

// ---- host diagnostics ------------------------------------------------------------
// Cullum-Willoughby ghost test (Eq. 25) and cluster weights (L270), cumulative spectral weight
// (Eq. 23).  T^(1) is T without its first row and column; l_k = min_j |theta_k - theta^(1)_j|; a Ritz value is
// flagged when l_k < tau = C_tau u_FP32 (theta_max - theta_min).  Ritz values closer than tau (chains of them) form
// one cluster, whose weight is the sum of its members' weights.
extern "C" int ftlm_ghost_diagnostic(int m, const double* alpha, const double* beta, double C_tau, double* theta,
                                     double* weight, double* ell, int* ghost, int* cluster, double* cluster_weight,
                                     double* F, double* tau_out) {
  if (m < 1 || !alpha || (m > 1 && !beta) || !theta || !weight || !(C_tau > 0.0)) {
    ftlm_set_error("ftlm_ghost_diagnostic: bad argument"); return FTLM_EINVAL;
  }
  int rc = ftlm_tridiag_eig(m, alpha, beta, theta, weight);
  if (rc != FTLM_OK) return rc;
  std::vector<double> th1((size_t)(m > 1 ? m - 1 : 0)), w1(th1.size());
  if (m > 1) {
    rc = ftlm_tridiag_eig(m - 1, alpha + 1, beta + 1, th1.data(), w1.data());
    if (rc != FTLM_OK) return rc;
  }
  const double tau = C_tau * 5.9604644775390625e-8 * (theta[m - 1] - theta[0]);
  if (tau_out) *tau_out = tau;
  size_t j = 0;                                          // both lists ascend: the nearest theta^(1) moves forward only
  for (int k = 0; k < m; ++k) {
    double l = INFINITY;
    if (m > 1) {
      while (j + 1 < th1.size() && th1[j + 1] <= theta[k]) ++j;
      l = std::fabs(theta[k] - th1[j]);
      if (j + 1 < th1.size()) l = std::min(l, std::fabs(theta[k] - th1[j + 1]));
    }
    if (ell) ell[k] = l;
    if (ghost) ghost[k] = l < tau ? 1 : 0;
  }
  int id = 0, first = 0;
  double acc = 0.0, run = 0.0;
  for (int k = 0; k <= m; ++k) {
    if (k == m || (k > 0 && theta[k] - theta[k - 1] > tau)) {      // cluster [first, k) ends
      for (int q = first; q < k; ++q) { if (cluster) cluster[q] = id; if (cluster_weight) cluster_weight[q] = acc; }
      ++id; first = k; acc = 0.0;
    }
    if (k < m) { acc += weight[k]; run += weight[k]; if (F) F[k] = run; }
  }
  return FTLM_OK;
}

// Eq. 22 (L225-L228): mean and population standard deviation over N_s seed sets, per temperature.
extern "C" int ftlm_sigma_emp(int n_seeds, int nT, const double* samples, double* mean, double* sigma) {
  if (n_seeds < 1 || nT < 0 || (nT > 0 && (!samples || !mean || !sigma))) { ftlm_set_error("ftlm_sigma_emp: bad argument"); return FTLM_EINVAL; }
  for (int i = 0; i < nT; ++i) {
    double s = 0.0;
    for (int q = 0; q < n_seeds; ++q) s += samples[(size_t)q * nT + i];
    const double mu = s / n_seeds;
    double v = 0.0;
    for (int q = 0; q < n_seeds; ++q) { const double d = samples[(size_t)q * nT + i] - mu; v += d * d; }
    mean[i] = mu;
    sigma[i] = std::sqrt(v / n_seeds);
  }
  return FTLM_OK;
}

// L230: sigma_theo = |O| / sqrt(Z_eff), Z_eff = Tr exp(-(H - E_0)/T)  (ftlm_thermo's Zs).
extern "C" int ftlm_sigma_theo(int nT, const double* O, const double* Z_eff, double* sigma) {
  if (nT < 0 || (nT > 0 && (!O || !Z_eff || !sigma))) { ftlm_set_error("ftlm_sigma_theo: bad argument"); return FTLM_EINVAL; }
  for (int i = 0; i < nT; ++i) {
    if (!(Z_eff[i] > 0.0)) { ftlm_set_error("ftlm_sigma_theo: Z_eff[%d] <= 0", i); return FTLM_EINVAL; }
    sigma[i] = std::fabs(O[i]) / std::sqrt(Z_eff[i]);
  }
  return FTLM_OK;
}
