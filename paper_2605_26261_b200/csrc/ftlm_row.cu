// ROW kernels: one thread per sector row, every row unranked, per-bond loop.  This is the
// paper's launch shape ("assigning one GPU thread to each
// sector-basis state") written for sm_100a; it is the plain in-library baseline and the path
// used for index-map queries.  The B200 design proper is in ftlm_tml.cu / ftlm_tmlr.cu / ftlm_passb.cu.
#define FTLM_TU 2
#include "ftlm_common.cuh"
#include "ftlm_index.cuh"

namespace {

struct RowParams {
  int N, K, nb, mode;
  int lin_h;
  const uint64_t* lin_hi;
  const uint32_t* lin_lo;
  int64_t dim;
  const void* binom;       // I[(N+1)*(K+1)]
  const BondDev* bonds;
  const uint2* clt;
  double diag0;
  // fused part
  ChainState* st;
  double* partials;
  unsigned int* ticket;
  int stride;
};

template <typename R> struct BondS { uint64_t mask; R Jh, Jq; int i, j; };

template <typename R, typename L, typename I>
__device__ __forceinline__ void load_tables(const RowParams& p, I* s_binom, BondS<R>* s_bonds) {
  const int nbin = (p.N + 1) * (p.K + 1);
  const I* g = (const I*)p.binom;
  for (int k = threadIdx.x; k < nbin; k += blockDim.x) ST_S(&s_binom[k], LD_G(&g[k]));
  for (int k = threadIdx.x; k < p.nb; k += blockDim.x) {
    const BondDev b = LD_G(&p.bonds[k]);
    BondS<R> sb;
    sb.mask = b.mask; sb.Jh = (R)b.Jh; sb.Jq = (R)b.Jq; sb.i = b.i; sb.j = b.j;
    ST_S(&s_bonds[k], sb);
  }
  __syncthreads();
}

// B > 1: the paper's batched Lanczos (L207, L309): B chains on interleaved vectors v[t][B] share the row state and
// every index computation; each chain's arithmetic is the B = 1 arithmetic in the same order (bit-identical results).
template <typename R, typename L, typename I, int MODE, bool FUSED, int B>
__global__ void __launch_bounds__(256)
hv_row_kernel(RowParams p, const R* __restrict__ v, const R* __restrict__ qprev, R* __restrict__ y) {
  FTLM_DYN_SMEM(smem);
  __shared__ double sh_red[96];
  if (FUSED) {
    bool all_done = true;
#pragma unroll
    for (int c = 0; c < B; ++c) all_done = all_done && p.st[c].done;
    if (all_done) return;
  }
  I* s_binom = (I*)smem;
  const int nbin = (p.N + 1) * (p.K + 1);
  BondS<R>* s_bonds = (BondS<R>*)(smem + (((size_t)nbin * sizeof(I) + 15) & ~(size_t)15));
  load_tables<R, L, I>(p, s_binom, s_bonds);
  const int K1 = p.K + 1;
  R bprev[B];
#pragma unroll
  for (int c = 0; c < B; ++c) bprev[c] = FUSED ? (R)p.st[c].beta_prev : (R)0;
  double s_qy[B], s_yy[B], s_qq[B];
#pragma unroll
  for (int c = 0; c < B; ++c) { s_qy[c] = 0.0; s_yy[c] = 0.0; s_qq[c] = 0.0; }
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < p.dim; t += stride) {
    const L n = unrank<L, I>((I)t, p.N, K1, p.K, s_binom);
    R acc[B], danti = 0;
#pragma unroll
    for (int c = 0; c < B; ++c) acc[c] = 0;
    for (int b = 0; b < p.nb; ++b) {
      const L m = (L)s_bonds[b].mask;
      const L x = n & m;
      if (x != 0 && x != m) {                                   // antiparallel spins
        I idx;
        if (MODE == FTLM_INDEX_CLT) idx = (I)clt_lookup((uint32_t)(n ^ m), p.clt);
        else if (MODE == FTLM_INDEX_LIN) idx = (I)lin_lookup((uint64_t)(n ^ m), p.lin_h, p.lin_hi, p.lin_lo);
        else idx = (I)t + cr_delta<L, I>(n, s_bonds[b].i, s_bonds[b].j, K1, s_binom);
#pragma unroll
        for (int c = 0; c < B; ++c) acc[c] += s_bonds[b].Jh * LDG(&v[(size_t)idx * B + c]);
        danti += s_bonds[b].Jq;
      }
    }
#pragma unroll
    for (int c = 0; c < B; ++c) {
      const R vt = LD_G(&v[(size_t)t * B + c]);
      R out = ((R)p.diag0 - 2 * danti) * vt + acc[c];
      if (FUSED) {
        out -= bprev[c] * LD_G(&qprev[(size_t)t * B + c]);
        s_qy[c] += (double)vt * (double)out;
        s_yy[c] += (double)out * (double)out;
        s_qq[c] += (double)vt * (double)vt;
      }
      ST_G(&y[(size_t)t * B + c], out);
    }
  }
  if (FUSED) {
#pragma unroll
    for (int c = 0; c < B; ++c)        // chain c: partials [3c .. 3c+3) x stride, ticket c, state c
      lanczos_finish(s_qy[c], s_yy[c], s_qq[c], p.partials + (size_t)3 * c * p.stride, p.stride, p.ticket + c, p.st + c, sh_red);
  }
}

// ---- ROWG: unrank once, then Gosper-style successor (north_star: "row bit-states by unranking plus Gosper-style
// successor enumeration"; L136 for the unrank) ---------------------------------------------------------------------
// A thread owns G = 8 consecutive rows: the label of the first comes from the inverse map, the next seven from the
// same-popcount successor  c = n & -n, r = n + c, n' = r | (((n ^ r) >> 2) >> ctz(n))  (the next larger integer with
// the same number of ones = the next basis state in ascending order, reading 2).  A lane's 8 rows are 32 (FP32) or
// 64 (FP64) contiguous bytes, a warp's 256 rows one contiguous kilobyte: the streams of v, q_prev and y stay fully
// coalesced while the N-step unrank is paid once per 8 rows.
#define ROWG_G 8
template <typename L>
__device__ __forceinline__ L gosper_next(L n) {
  const L c = n & (L)(0 - n);
  const L r = n + c;
  return r | (((n ^ r) >> 2) >> (ffs_(n) - 1));
}

template <typename R, typename L, typename I, int MODE, bool FUSED>
__global__ void __launch_bounds__(256)
hv_rowg_kernel(RowParams p, const R* __restrict__ v, const R* __restrict__ qprev, R* __restrict__ y) {
  FTLM_DYN_SMEM(smem);
  __shared__ double sh_red[96];
  if (FUSED) { if (p.st->done) return; }
  I* s_binom = (I*)smem;
  const int nbin = (p.N + 1) * (p.K + 1);
  BondS<R>* s_bonds = (BondS<R>*)(smem + (((size_t)nbin * sizeof(I) + 15) & ~(size_t)15));
  load_tables<R, L, I>(p, s_binom, s_bonds);
  const int K1 = p.K + 1;
  const R bprev = FUSED ? (R)p.st->beta_prev : (R)0;
  double s_qy = 0.0, s_yy = 0.0, s_qq = 0.0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x * ROWG_G;
  for (int64_t t0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * ROWG_G; t0 < p.dim; t0 += stride) {
    const int ng = (int)(p.dim - t0 < ROWG_G ? p.dim - t0 : ROWG_G);
    R vt[ROWG_G], qp[ROWG_G], out[ROWG_G];
#pragma unroll
    for (int g = 0; g < ROWG_G; ++g) {
      vt[g] = g < ng ? LD_G(&v[t0 + g]) : (R)0;
      qp[g] = (FUSED && g < ng) ? LD_G(&qprev[t0 + g]) : (R)0;
    }
    L n = unrank<L, I>((I)t0, p.N, K1, p.K, s_binom);
#pragma unroll
    for (int g = 0; g < ROWG_G; ++g) {                             // unrolled: the 8 rows' values stay in registers
      if (g >= ng) break;
      const int64_t t = t0 + g;
      R acc = 0, danti = 0;
      for (int b = 0; b < p.nb; ++b) {
        const L m = (L)s_bonds[b].mask;
        const L x = n & m;
        if (x != 0 && x != m) {                                   // antiparallel spins
          I idx;
          if (MODE == FTLM_INDEX_CLT) idx = (I)clt_lookup((uint32_t)(n ^ m), p.clt);
          else if (MODE == FTLM_INDEX_LIN) idx = (I)lin_lookup((uint64_t)(n ^ m), p.lin_h, p.lin_hi, p.lin_lo);
          else idx = (I)t + cr_delta<L, I>(n, s_bonds[b].i, s_bonds[b].j, K1, s_binom);
          acc += s_bonds[b].Jh * LDG(&v[idx]);
          danti += s_bonds[b].Jq;
        }
      }
      R o = ((R)p.diag0 - 2 * danti) * vt[g] + acc;
      if (FUSED) {
        o -= bprev * qp[g];
        s_qy += (double)vt[g] * (double)o;
        s_yy += (double)o * (double)o;
        s_qq += (double)vt[g] * (double)vt[g];
      }
      out[g] = o;
      if (n != 0) n = gosper_next<L>(n);                          // (n == 0: the one-state sector N_up = 0)
    }
#pragma unroll
    for (int g = 0; g < ROWG_G; ++g) if (g < ng) ST_G(&y[t0 + g], out[g]);
  }
  if (FUSED) lanczos_finish(s_qy, s_yy, s_qq, p.partials, p.stride, p.ticket, p.st, sh_red);
}

// neighbour indices through the same enumeration (unrank at the first row of a group, successor afterwards)
template <typename L, typename I, int MODE>
__global__ void __launch_bounds__(256)
neighbors_rowg_kernel(RowParams p, int64_t row0, int64_t nrows, int64_t* __restrict__ out) {
  FTLM_DYN_SMEM(smem);
  I* s_binom = (I*)smem;
  const int nbin = (p.N + 1) * (p.K + 1);
  BondS<float>* s_bonds = (BondS<float>*)(smem + (((size_t)nbin * sizeof(I) + 15) & ~(size_t)15));
  load_tables<float, L, I>(p, s_binom, s_bonds);
  const int K1 = p.K + 1;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x * ROWG_G;
  for (int64_t r0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * ROWG_G; r0 < nrows; r0 += stride) {
    L n = unrank<L, I>((I)(row0 + r0), p.N, K1, p.K, s_binom);
    for (int g = 0; g < ROWG_G && r0 + g < nrows; ++g) {
      const int64_t t = row0 + r0 + g;
      for (int b = 0; b < p.nb; ++b) {
        const L m = (L)s_bonds[b].mask;
        const L x = n & m;
        int64_t idx = -1;
        if (x != 0 && x != m) {
          if (MODE == FTLM_INDEX_CLT) idx = (int64_t)clt_lookup((uint32_t)(n ^ m), p.clt);
          else if (MODE == FTLM_INDEX_LIN) idx = (int64_t)lin_lookup((uint64_t)(n ^ m), p.lin_h, p.lin_hi, p.lin_lo);
          else idx = (int64_t)(I)((I)t + cr_delta<L, I>(n, s_bonds[b].i, s_bonds[b].j, K1, s_binom));
        }
        ST_G(&out[(r0 + g) * p.nb + b], idx);
      }
      if (n != 0) n = gosper_next<L>(n);
    }
  }
}

template <typename L, typename I, int MODE>
__global__ void __launch_bounds__(256)
neighbors_row_kernel(RowParams p, int64_t row0, int64_t nrows, int64_t* __restrict__ out) {
  FTLM_DYN_SMEM(smem);
  I* s_binom = (I*)smem;
  const int nbin = (p.N + 1) * (p.K + 1);
  BondS<float>* s_bonds = (BondS<float>*)(smem + (((size_t)nbin * sizeof(I) + 15) & ~(size_t)15));
  load_tables<float, L, I>(p, s_binom, s_bonds);
  const int K1 = p.K + 1;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < nrows; r += stride) {
    const int64_t t = row0 + r;
    const L n = unrank<L, I>((I)t, p.N, K1, p.K, s_binom);
    for (int b = 0; b < p.nb; ++b) {
      const L m = (L)s_bonds[b].mask;
      const L x = n & m;
      int64_t idx = -1;
      if (x != 0 && x != m) {
        if (MODE == FTLM_INDEX_CLT) idx = (int64_t)clt_lookup((uint32_t)(n ^ m), p.clt);
        else if (MODE == FTLM_INDEX_LIN) idx = (int64_t)lin_lookup((uint64_t)(n ^ m), p.lin_h, p.lin_hi, p.lin_lo);
        else idx = (int64_t)(I)((I)t + cr_delta<L, I>(n, s_bonds[b].i, s_bonds[b].j, K1, s_binom));
      }
      ST_G(&out[r * p.nb + b], idx);
    }
  }
}

template <typename L, typename I>
__global__ void index_of_kernel(RowParams p, const uint64_t* __restrict__ labels, int64_t n,
                                int64_t* __restrict__ out) {
  FTLM_DYN_SMEM(smem);
  I* s_binom = (I*)smem;
  const int nbin = (p.N + 1) * (p.K + 1);
  for (int k = threadIdx.x; k < nbin; k += blockDim.x) ST_S(&s_binom[k], LD_G(&((const I*)p.binom)[k]));
  __syncthreads();
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += stride) {
    const uint64_t lab = LD_G(&labels[k]);
    int64_t idx;
    if (p.mode == FTLM_INDEX_CLT) {
      idx = clt_lookup_checked(lab, p.N, p.clt);
    } else if (p.mode == FTLM_INDEX_LIN) {
      const bool in = (lab >> p.N) == 0 && __popcll(lab) == p.K;          // N <= 48 in this mode
      idx = in ? (int64_t)lin_lookup(lab, p.lin_h, p.lin_hi, p.lin_lo) : -1;
    } else {
      const bool in = (p.N >= 64 || (lab >> p.N) == 0) && __popcll(lab) == p.K;
      idx = in ? (int64_t)rank_alg1<L, I>((L)lab, p.N, p.K + 1, p.K, s_binom) : -1;
    }
    ST_G(&out[k], idx);
  }
}

template <typename L, typename I>
__global__ void state_of_kernel(RowParams p, const int64_t* __restrict__ idx, int64_t n,
                                uint64_t* __restrict__ out) {
  FTLM_DYN_SMEM(smem);
  I* s_binom = (I*)smem;
  const int nbin = (p.N + 1) * (p.K + 1);
  for (int k = threadIdx.x; k < nbin; k += blockDim.x) ST_S(&s_binom[k], LD_G(&((const I*)p.binom)[k]));
  __syncthreads();
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += stride) {
    const int64_t t = LD_G(&idx[k]);
    ST_G(&out[k], (t < 0 || t >= p.dim) ? ~0ull : (uint64_t)unrank<L, I>((I)t, p.N, p.K + 1, p.K, s_binom));
  }
}

RowParams make_params(ftlm_ctx* c) {
  RowParams p;
  p.N = c->N; p.K = c->N_up; p.nb = c->nb; p.mode = c->mode; p.dim = c->dim;
  p.binom = c->idx64 ? (const void*)c->d_binom64 : (const void*)c->d_binom32;
  p.bonds = c->d_bonds; p.clt = c->d_clt; p.diag0 = c->diag0;
  p.lin_h = c->lin_h; p.lin_hi = c->d_lin_hi; p.lin_lo = c->d_lin_lo;
  p.st = c->d_state; p.partials = c->d_partials; p.ticket = c->d_ticket; p.stride = c->max_blocks;
  return p;
}

size_t table_smem(const ftlm_ctx* c, size_t bond_sz) {
  const size_t isz = c->idx64 ? 8 : 4;
  size_t b = ((size_t)(c->N + 1) * (c->N_up + 1) * isz + 15) & ~(size_t)15;
  return b + (size_t)c->nb * bond_sz;
}

int grid_for(const ftlm_ctx* c, int64_t work, int per_sm) {
  int64_t blocks = (work + 255) / 256;
  int64_t cap = (int64_t)c->sm_count * per_sm;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  return (int)blocks;
}

template <typename R, typename L, typename I>
int launch_hv(ftlm_ctx* c, const RowParams& p, const void* v, const void* qp, void* y, int fused, int batch,
              cudaStream_t s) {
  const size_t sm = table_smem(c, sizeof(BondS<R>));
  const int grid = grid_for(c, c->dim, 8);
  if (fused && grid > c->max_blocks) { ftlm_set_error("internal: grid > max_blocks"); return FTLM_EINVAL; }
  if (batch != 1 && !fused) { ftlm_set_error("ROW: batched vectors exist in the fused Lanczos step only"); return FTLM_EINVAL; }
#define LAUNCH(MODE, FUSED, BB)                                                                  \
  do {                                                                                           \
    auto k = hv_row_kernel<R, L, I, MODE, FUSED, BB>;                                            \
    if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); \
    FTLM_LAUNCH(k, grid, 256, sm, s, p, (const R*)v, (const R*)qp, (R*)y);                                \
  } while (0)
#define LAUNCHB(MODE)                                                                            \
  do {                                                                                           \
    if (!fused) LAUNCH(MODE, false, 1);                                                          \
    else if (batch == 1) LAUNCH(MODE, true, 1);                                                  \
    else if (batch == 2) LAUNCH(MODE, true, 2);                                                  \
    else if (batch == 4) LAUNCH(MODE, true, 4);                                                  \
    else { ftlm_set_error("ROW: batch must be 1, 2 or 4 (got %d)", batch); return FTLM_EINVAL; } \
  } while (0)
  if (c->mode == FTLM_INDEX_CLT) LAUNCHB(FTLM_INDEX_CLT); else if (c->mode == FTLM_INDEX_LIN) LAUNCHB(FTLM_INDEX_LIN); else LAUNCHB(FTLM_INDEX_CR);
#undef LAUNCHB
#undef LAUNCH
  CK(cudaGetLastError());
  return FTLM_OK;
}

}  // namespace

int ftlm_launch_hv_row(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, int batch, cudaStream_t s) {
  RowParams p = make_params(c);
  if (c->prec == FTLM_FP32) {
    if (!c->lab64) return launch_hv<float, uint32_t, uint32_t>(c, p, v, qprev, y, fused, batch, s);
    if (!c->idx64) return launch_hv<float, uint64_t, uint32_t>(c, p, v, qprev, y, fused, batch, s);
    return launch_hv<float, uint64_t, uint64_t>(c, p, v, qprev, y, fused, batch, s);
  } else {
    if (!c->lab64) return launch_hv<double, uint32_t, uint32_t>(c, p, v, qprev, y, fused, batch, s);
    if (!c->idx64) return launch_hv<double, uint64_t, uint32_t>(c, p, v, qprev, y, fused, batch, s);
    return launch_hv<double, uint64_t, uint64_t>(c, p, v, qprev, y, fused, batch, s);
  }
}

namespace {
template <typename R, typename L, typename I>
int launch_hv_g(ftlm_ctx* c, const RowParams& p, const void* v, const void* qp, void* y, int fused, cudaStream_t s) {
  const size_t sm = table_smem(c, sizeof(BondS<R>));
  const int grid = grid_for(c, (c->dim + ROWG_G - 1) / ROWG_G, 8);
  if (fused && grid > c->max_blocks) { ftlm_set_error("internal: grid > max_blocks"); return FTLM_EINVAL; }
#define LAUNCHG(MODE, FUSED)                                                                     \
  do {                                                                                           \
    auto k = hv_rowg_kernel<R, L, I, MODE, FUSED>;                                               \
    if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); \
    FTLM_LAUNCH(k, grid, 256, sm, s, p, (const R*)v, (const R*)qp, (R*)y);                                \
  } while (0)
  if (c->mode == FTLM_INDEX_CLT) { if (fused) LAUNCHG(FTLM_INDEX_CLT, true); else LAUNCHG(FTLM_INDEX_CLT, false); }
  else if (c->mode == FTLM_INDEX_LIN) { if (fused) LAUNCHG(FTLM_INDEX_LIN, true); else LAUNCHG(FTLM_INDEX_LIN, false); }
  else { if (fused) LAUNCHG(FTLM_INDEX_CR, true); else LAUNCHG(FTLM_INDEX_CR, false); }
#undef LAUNCHG
  CK(cudaGetLastError());
  return FTLM_OK;
}
}  // namespace

int ftlm_launch_hv_rowg(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, cudaStream_t s) {
  RowParams p = make_params(c);
  if (c->prec == FTLM_FP32) {
    if (!c->lab64) return launch_hv_g<float, uint32_t, uint32_t>(c, p, v, qprev, y, fused, s);
    if (!c->idx64) return launch_hv_g<float, uint64_t, uint32_t>(c, p, v, qprev, y, fused, s);
    return launch_hv_g<float, uint64_t, uint64_t>(c, p, v, qprev, y, fused, s);
  } else {
    if (!c->lab64) return launch_hv_g<double, uint32_t, uint32_t>(c, p, v, qprev, y, fused, s);
    if (!c->idx64) return launch_hv_g<double, uint64_t, uint32_t>(c, p, v, qprev, y, fused, s);
    return launch_hv_g<double, uint64_t, uint64_t>(c, p, v, qprev, y, fused, s);
  }
}

int ftlm_launch_neighbors_rowg(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s) {
  RowParams p = make_params(c);
  const size_t sm = table_smem(c, sizeof(BondS<float>));
  const int grid = grid_for(c, (nrows + ROWG_G - 1) / ROWG_G, 8);
#define LAUNCHNG(L, I)                                                                                \
  do {                                                                                                \
    if (c->mode == FTLM_INDEX_CLT) { auto k = neighbors_rowg_kernel<L, I, FTLM_INDEX_CLT>; if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); FTLM_LAUNCH(k, grid, 256, sm, s, p, row0, nrows, d_idx); } \
    else if (c->mode == FTLM_INDEX_LIN) { auto k = neighbors_rowg_kernel<L, I, FTLM_INDEX_LIN>; if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); FTLM_LAUNCH(k, grid, 256, sm, s, p, row0, nrows, d_idx); } \
    else { auto k = neighbors_rowg_kernel<L, I, FTLM_INDEX_CR>; if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); FTLM_LAUNCH(k, grid, 256, sm, s, p, row0, nrows, d_idx); } \
  } while (0)
  if (!c->lab64) LAUNCHNG(uint32_t, uint32_t);
  else if (!c->idx64) LAUNCHNG(uint64_t, uint32_t);
  else LAUNCHNG(uint64_t, uint64_t);
#undef LAUNCHNG
  CK(cudaGetLastError());
  return FTLM_OK;
}

int ftlm_launch_neighbors_row(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s) {
  RowParams p = make_params(c);
  const size_t sm = table_smem(c, sizeof(BondS<float>));
  const int grid = grid_for(c, nrows, 8);
#define LAUNCHN(L, I)                                                                                 \
  do {                                                                                                \
    if (c->mode == FTLM_INDEX_CLT) {                                                                  \
      auto k = neighbors_row_kernel<L, I, FTLM_INDEX_CLT>;                                            \
      if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); \
      FTLM_LAUNCH(k, grid, 256, sm, s, p, row0, nrows, d_idx);                                                 \
    } else if (c->mode == FTLM_INDEX_LIN) {                                                           \
      auto k = neighbors_row_kernel<L, I, FTLM_INDEX_LIN>;                                            \
      if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); \
      FTLM_LAUNCH(k, grid, 256, sm, s, p, row0, nrows, d_idx);                                                 \
    } else {                                                                                          \
      auto k = neighbors_row_kernel<L, I, FTLM_INDEX_CR>;                                             \
      if (sm > 48 * 1024) CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)); \
      FTLM_LAUNCH(k, grid, 256, sm, s, p, row0, nrows, d_idx);                                                 \
    }                                                                                                 \
  } while (0)
  if (!c->lab64) LAUNCHN(uint32_t, uint32_t);
  else if (!c->idx64) LAUNCHN(uint64_t, uint32_t);
  else LAUNCHN(uint64_t, uint64_t);
#undef LAUNCHN
  CK(cudaGetLastError());
  return FTLM_OK;
}

extern "C" int ftlm_index_of(ftlm_ctx* c, const uint64_t* d_labels, int64_t n, int64_t* d_idx, void* stream) {
  if (!c || (n > 0 && (!d_labels || !d_idx)) || n < 0) { ftlm_set_error("ftlm_index_of: bad argument"); return FTLM_EINVAL; }
  if (n == 0) return FTLM_OK;
  CK(cudaSetDevice(c->device));
  RowParams p = make_params(c);
  const size_t sm = table_smem(c, 0);
  const int grid = grid_for(c, n, 8);
  cudaStream_t s = (cudaStream_t)stream;
  ftlm_chk_caller(s, d_labels, (size_t)n * 8); ftlm_chk_caller(s, d_idx, (size_t)n * 8);
  if (!c->lab64) { auto k__ = index_of_kernel<uint32_t, uint32_t>; FTLM_LAUNCH(k__, grid, 256, sm, s, p, d_labels, n, d_idx); }
  else if (!c->idx64) { auto k__ = index_of_kernel<uint64_t, uint32_t>; FTLM_LAUNCH(k__, grid, 256, sm, s, p, d_labels, n, d_idx); }
  else { auto k__ = index_of_kernel<uint64_t, uint64_t>; FTLM_LAUNCH(k__, grid, 256, sm, s, p, d_labels, n, d_idx); }
  CK(cudaGetLastError());
  return FTLM_OK;
}

extern "C" int ftlm_state_of(ftlm_ctx* c, const int64_t* d_idx, int64_t n, uint64_t* d_labels, void* stream) {
  if (!c || (n > 0 && (!d_labels || !d_idx)) || n < 0) { ftlm_set_error("ftlm_state_of: bad argument"); return FTLM_EINVAL; }
  if (n == 0) return FTLM_OK;
  CK(cudaSetDevice(c->device));
  RowParams p = make_params(c);
  const size_t sm = table_smem(c, 0);
  const int grid = grid_for(c, n, 8);
  cudaStream_t s = (cudaStream_t)stream;
  ftlm_chk_caller(s, d_labels, (size_t)n * 8); ftlm_chk_caller(s, d_idx, (size_t)n * 8);
  if (!c->lab64) { auto k__ = state_of_kernel<uint32_t, uint32_t>; FTLM_LAUNCH(k__, grid, 256, sm, s, p, d_idx, n, d_labels); }
  else if (!c->idx64) { auto k__ = state_of_kernel<uint64_t, uint32_t>; FTLM_LAUNCH(k__, grid, 256, sm, s, p, d_idx, n, d_labels); }
  else { auto k__ = state_of_kernel<uint64_t, uint64_t>; FTLM_LAUNCH(k__, grid, 256, sm, s, p, d_idx, n, d_labels); }
  CK(cudaGetLastError());
  return FTLM_OK;
}
