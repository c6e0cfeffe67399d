// ftlm_autotune - choose the H.v kernel configuration of a handle by measurement, on the device.
//
// Every candidate (ROW, TILE, TML with its bonds that leave the tile read from global memory, TML +
// PASS-B windows in several window sizes, with the TML or the TMLR in-tile pass) first computes y = H v for one seeded random vector and is
// compared, on the device, with the ROW kernel's result (the paper's launch shape, thread per row,
// Eq. 12 / Alg. 1 / Alg. 2 directly): a candidate whose norm-relative deviation exceeds the
// north_star tolerance (1e-5 FP32, 1e-12 FP64) is rejected; so is one whose first three fused Lanczos steps
// (alpha_1..3, beta_1..2) differ from the ROW kernel's by more than 1e-4 (FP32) / 1e-9 (FP64).  The valid
// candidates are timed with CUDA events over `reps` whole fused steps and the fastest is left selected.  All arithmetic
// is in the library's kernels; nothing here runs on the CPU.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#define FTLM_TU 6
#include "ftlm_common.cuh"

namespace {

// out[0] += sum (a - ref)^2, out[1] += sum ref^2, out[2] = max |a - ref|, out[3] = max |v|  (the last two as the
// bit patterns of non-negative doubles, which order like unsigned integers)
template <typename R>
__global__ void __launch_bounds__(256)
diff_norm_kernel(const R* __restrict__ a, const R* __restrict__ ref, const R* __restrict__ v, int64_t n, double* __restrict__ out) {
  double d2 = 0.0, r2 = 0.0, dmax = 0.0, vmax = 0.0;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
    const double x = (double)LD_G(&a[k]), y = (double)LD_G(&ref[k]);
    double d = fabs(x - y);
    if (!(d == d)) d = 1e300;                          // a NaN in the candidate counts as a huge deviation
    d2 += d < 1e150 ? d * d : 1e300;
    r2 += y * y;
    dmax = fmax(dmax, d);
    vmax = fmax(vmax, fabs((double)LD_G(&v[k])));
  }
  d2 = warp_sum(d2);
  r2 = warp_sum(r2);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    dmax = fmax(dmax, __shfl_down_sync(0xffffffffu, dmax, o));
    vmax = fmax(vmax, __shfl_down_sync(0xffffffffu, vmax, o));
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&out[0], d2); atomicAdd(&out[1], r2);
    atomicMax((unsigned long long*)&out[2], (unsigned long long)__double_as_longlong(dmax));
    atomicMax((unsigned long long*)&out[3], (unsigned long long)__double_as_longlong(vmax));
  }
}

struct Cand {
  const char* name;
  int kernel, passb, smax, ctas, tmlr, lazy, split;   // split: w | m << 8 of the TML tile (0 = auto)
  int verified;   // 1: this configuration has a green -m gpu parity record on a B200 in its present source form
                  // (checked build with zero violations, then the release build); see DESIGN.md section 13.
                  // Others are run only after ftlm_set_option(ctx, "allow_unverified", 1).
};

// home_split: the split the handle had when tuning began (candidates with split == 0 keep it)
int apply_cand(ftlm_ctx* c, const Cand& k, int home_split) {
  int rc;
  if (k.kernel == FTLM_KERNEL_TML) {
    const int want = k.split ? k.split : home_split;
    if ((c->tml_low_bits | (c->tml_mid_bits << 8)) != want && (rc = ftlm_set_option(c, "tml_split", want)) != FTLM_OK) return rc;
    if ((rc = ftlm_set_option(c, "passb_smax", k.smax)) != FTLM_OK) return rc;
    if ((rc = ftlm_set_option(c, "passb_ctas", k.ctas)) != FTLM_OK) return rc;
    if ((rc = ftlm_set_option(c, "passb", k.passb)) != FTLM_OK) return rc;
  }
  if ((rc = ftlm_set_option(c, "tmlr", k.tmlr)) != FTLM_OK) return rc;
  if ((rc = ftlm_set_option(c, "lazy_norm", k.lazy)) != FTLM_OK) return rc;
  return ftlm_set_option(c, "kernel", k.kernel);
}

}  // namespace

extern "C" int ftlm_autotune(ftlm_ctx* c, int reps, char* report, int report_cap, void* stream) {
  if (!c || reps < 1) { ftlm_set_error("ftlm_autotune: bad argument"); return FTLM_EINVAL; }
  CK(cudaSetDevice(c->device));
  cudaStream_t s = (cudaStream_t)stream;
  const size_t esz = ftlm_elem_size(c), bytes = (size_t)c->dim * esz;
  void *v = nullptr, *yref = nullptr, *y = nullptr;
  double* d_out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  std::string rep = "[";
  int rc = FTLM_OK;
  auto cleanup = [&]() {
    ftlm_dfree(v); ftlm_dfree(yref); ftlm_dfree(y); ftlm_dfree(d_out);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
  };
  if (ftlm_dmalloc(&v, bytes) != cudaSuccess || ftlm_dmalloc(&yref, bytes) != cudaSuccess || ftlm_dmalloc(&y, bytes) != cudaSuccess ||
      ftlm_dmalloc((void**)&d_out, 32) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
    cudaGetLastError(); cleanup();
    ftlm_set_error("ftlm_autotune: cannot allocate 3 x %zu bytes", bytes);
    return FTLM_ENOMEM;
  }
  const int saved_kernel = c->kernel, saved_pb = c->use_passb, saved_smax = c->passb_smax, saved_ctas = c->passb_ctas, saved_tmlr = c->use_tmlr, saved_lazy = c->lazy_norm,
            saved_w = c->tml_low_bits, saved_m = c->tml_mid_bits;
  const int home_split = saved_w | (saved_m << 8);
  const Cand cands[] = {
      {"row", FTLM_KERNEL_ROW, 0, 0, 0, 0, 0, 0, 1},
      {"rowg", FTLM_KERNEL_ROWG, 0, 0, 0, 0, 0, 0, 0},
      {"tml", FTLM_KERNEL_TML, 0, 0, 0, 0, 0, 0, 0},
      {"tml+passb", FTLM_KERNEL_TML, 1, 0, 0, 0, 0, 0, 0},
      {"tml+passb_1cta", FTLM_KERNEL_TML, 1, 0, 1, 0, 0, 0, 0},
      {"tml+passb_s11", FTLM_KERNEL_TML, 1, 11, 0, 0, 0, 0, 0},
      {"tml+passb_s10", FTLM_KERNEL_TML, 1, 10, 0, 0, 0, 0, 0},
      {"tmlr+passb", FTLM_KERNEL_TML, 1, 0, 0, 1, 0, 0, 0},
      {"tmlr+passb_s11", FTLM_KERNEL_TML, 1, 11, 0, 1, 0, 0, 0},
      {"tmlr+passb_lazy", FTLM_KERNEL_TML, 1, 0, 0, 1, 1, 0, 0},
      {"tmlr+passb_s11_lazy", FTLM_KERNEL_TML, 1, 11, 0, 1, 1, 0, 0},
      {"tml_w9m7", FTLM_KERNEL_TML, 0, 0, 0, 0, 0, 9 | (7 << 8), 0},
      {"tml_w9m7+passb", FTLM_KERNEL_TML, 1, 0, 0, 0, 0, 9 | (7 << 8), 0},
  };
  const int ncand = (int)(sizeof(cands) / sizeof(cands[0]));
  const double tol = c->prec == FTLM_FP32 ? 1e-5 : 1e-12;
  double sumabsJ = 0.0;
  for (const BondDev& bd : c->bonds) sumabsJ += std::fabs(2.0 * bd.Jh);
  int best = -1;
  double best_ms = 0.0;
  // three fused Lanczos steps from the seeded start vector: alpha_1..3, beta_1..2 (host copies)
  auto fused_probe = [&](double* ab) -> int {
    double al[8] = {0}, be[8] = {0};
    int m_eff = 0;
    int r = ftlm_chain_begin(c, nullptr, 0x5EEDull, 0, s);
    if (r == FTLM_OK) r = ftlm_chain_steps(c, 3, s);
    if (r == FTLM_OK) r = ftlm_chain_end(c, al, be, 8, &m_eff, s);
    for (int k = 0; k < 3; ++k) ab[k] = al[k];
    for (int k = 0; k < 2; ++k) ab[3 + k] = be[k];
    return r;
  };
  double ab_ref[5] = {0, 0, 0, 0, 0};
  const double tol_f = c->prec == FTLM_FP32 ? 1e-4 : 1e-9;
  // reference: the ROW kernel on a seeded random vector, and its fused steps
  rc = ftlm_fill_random(c, 0x5EEDull, 0, v, s);
  if (rc == FTLM_OK) rc = apply_cand(c, cands[0], home_split);
  if (rc == FTLM_OK) rc = ftlm_apply_H(c, v, yref, s);
  if (rc == FTLM_OK) rc = fused_probe(ab_ref);
  for (int k = 0; k < ncand && rc == FTLM_OK; ++k) {
    const Cand& cd = cands[k];
    if (!cd.verified && !c->allow_unverified) continue;                              // never first contact with a device from here
    if (k > 0 && c->autotune_mask && !((c->autotune_mask >> k) & 1ull)) continue;    // the caller's selection (bench.py: those its checked pre-flight passed)
    if (apply_cand(c, cd, home_split) != FTLM_OK) continue;                          // not available for this sector
    if (cd.kernel == FTLM_KERNEL_TML && (!c->tml || (cd.passb && !c->passb) || (cd.tmlr && !c->tmlr) || (cd.lazy && !ftlm_tmlr_lazy_ok(c)))) continue;
    double h_out[4] = {0.0, 0.0, 0.0, 0.0};
    if (cudaMemsetAsync(d_out, 0, 32, s) != cudaSuccess) { rc = FTLM_ECUDA; break; }
    if ((rc = ftlm_apply_H(c, v, y, s)) != FTLM_OK) break;
    const int grid = c->sm_count * 8;
    if (c->prec == FTLM_FP32) { auto kk = diff_norm_kernel<float>; FTLM_LAUNCH(kk, grid, 256, 0, s, (const float*)y, (const float*)yref, (const float*)v, c->dim, d_out); }
    else { auto kk = diff_norm_kernel<double>; FTLM_LAUNCH(kk, grid, 256, 0, s, (const double*)y, (const double*)yref, (const double*)v, c->dim, d_out); }
    if (cudaMemcpyAsync(h_out, d_out, 32, cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess) {
      rc = ftlm_cuda_fail(cudaGetLastError(), "ftlm_autotune: candidate run"); break;
    }
    const double rel = h_out[1] > 0.0 ? std::sqrt(h_out[0] / h_out[1]) : (h_out[0] > 0.0 ? 1.0 : 0.0);
    // element-wise criterion beside the norm (a tile that drops one gather on a few rows moves the norm by < 1e-5):
    // two sequentially rounded sums of <= N_B + 1 products differ by at most 2 (N_B + 2) u sum|J_b| max|v|
    const double elem_bound = 2.0 * (c->nb + 2) * (c->prec == FTLM_FP32 ? 5.9604644775390625e-8 : 1.1102230246251565e-16) * (sumabsJ + std::fabs(c->h) * c->N / 2.0) * h_out[3];
    bool valid = rel <= tol && h_out[2] <= elem_bound;
    double dfused = 0.0;
    if (valid) {                                         // the fused step (recurrence, FP64 sums, finish) must agree too
      double ab[5];
      if ((rc = fused_probe(ab)) != FTLM_OK) break;
      for (int q = 0; q < 5; ++q) {
        const double d = std::fabs(ab[q] - ab_ref[q]) / std::fmax(1.0, std::fabs(ab_ref[q]));
        dfused = std::fmax(dfused, d == d ? d : 1e300);
      }
      valid = dfused <= tol_f;
    }
    float ms = 0.f;
    if (valid) {                                         // time `reps` whole fused steps (H.v passes + normalisation)
      if ((rc = ftlm_chain_begin(c, nullptr, 0x5EEDull, 0, s)) != FTLM_OK) break;
      if ((rc = ftlm_chain_steps(c, 1, s)) != FTLM_OK) break;
      cudaEventRecord(e0, s);
      rc = ftlm_chain_steps(c, reps, s);
      cudaEventRecord(e1, s);
      if (rc != FTLM_OK) break;
      if (cudaEventSynchronize(e1) != cudaSuccess) { rc = ftlm_cuda_fail(cudaGetLastError(), "ftlm_autotune: timing"); break; }
      cudaEventElapsedTime(&ms, e0, e1);
      ms /= (float)reps;
      if (best < 0 || ms < best_ms) { best = k; best_ms = ms; }
    }
    char line[384];
    snprintf(line, sizeof(line), "%s{\"name\": \"%s\", \"index\": %d, \"valid\": %s, \"relerr\": %.3e, \"maxabs\": %.3e, \"elem_bound\": %.3e, \"fused_dev\": %.3e, \"ms\": %.5f, \"windows\": %d}",
             rep.size() > 1 ? ", " : "", cd.name, k, valid ? "true" : "false", rel, h_out[2], elem_bound, dfused, (double)ms,
             (cd.kernel == FTLM_KERNEL_TML && c->passb) ? ftlm_passb_windows(c) : 0);
    rep += line;
  }
  rep += "]";
  if (rc == FTLM_OK && best >= 0) rc = apply_cand(c, cands[best], home_split);
  else {                                                                  // restore what the caller had
    c->passb_smax = saved_smax; c->passb_ctas = saved_ctas; c->use_tmlr = saved_tmlr; c->lazy_norm = saved_lazy;
    c->use_passb = saved_pb;
    ftlm_set_option(c, "tml_split", saved_w | (saved_m << 8));
    c->kernel = saved_kernel;
    if (rc == FTLM_OK) { ftlm_set_error("ftlm_autotune: no valid candidate"); rc = FTLM_EUNSUPPORTED; }
  }
  if (rc == FTLM_OK) { c->autotuned = best + 1; c->autotune_ms = best_ms; }
  if (report && report_cap > 0) {
    strncpy(report, rep.c_str(), (size_t)report_cap - 1);
    report[report_cap - 1] = 0;
  }
  cleanup();
  return rc;
}
