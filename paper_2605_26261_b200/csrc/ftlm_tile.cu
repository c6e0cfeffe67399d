// TILE kernels - the B200 design of the gather H.v.
//
// A label is split n = (H << w) | L.  All rows that share the high part H are consecutive
// ("run"): index = base(H) + lr(L), lr = rank of L among the w-bit words of equal popcount
// k = N_up - popc(H), base(H) = number of sector labels below H << w.  One CTA owns one run at
// a time, so everything that depends on H alone is CTA-uniform and computed once per run:
//   * bond inside L ("ll"):   neighbour stays in the run  -> gather from the run staged in smem
//   * bond inside H ("hh"):   antiparallel or not is uniform; the neighbour run has the same k
//                             and the same lr -> a coalesced stream v[base(H') + lr]
//   * bond across ("mixed"):  neighbour run H' = H ^ bit_j has k' = k +- 1; it is staged in smem
//                             once per high site j and gathered at lr(L ^ bit_i)
// Index strategies (both bit-exact with the ROW path and the oracle):
//   CR : base(H) by combinatorial ranking over the high bits (binomials in smem, Eq. 15-16 at
//        d = 2), lr(L) from a 2^w-entry chunk table generated from the same binomials - "rank
//        updated incrementally across the two flipped bit positions": an ll flip changes only
//        lr, an hh flip only base, a mixed flip both.
//   CLT: the (M_b, C_b) blocks of Alg. 2 covering a run are contiguous (2^(w-5) blocks); the
//        chunk of the own run and of each neighbour run is staged in smem and looked up there.
// Off-diagonal + diagonal are merged: y = diag0*v_t + sum_anti (J_b/2) (v[src] - v_t), because
// the diagonal loses 2*(J_b/4) = J_b/2 per antiparallel bond.
#include <algorithm>
#include <vector>

#include "ftlm_common.cuh"

#define TILE_THREADS 512
#define TILE_MAX_HH 128
#define TILE_MAX_SITES 32

struct TileLL { uint32_t mask; float pad; double Jh; };
struct TileHH { uint32_t mask; int pad; double Jh; };
struct TileMX { int site; int first; int count; int pad; };   // high site (position in H), slice of mx_low
struct TileMXLow { int bit; int pad; double Jh; };

struct TilePlan {
  int w = 0, nh = 0;                 // low bits, high bits
  int n_ll = 0, n_hh = 0, n_mx = 0, n_mxlow = 0;
  int max_run = 0;
  uint32_t n_H = 0;                  // 2^nh
  uint16_t* d_lr_tab = nullptr;      // [2^w]
  uint16_t* d_low_states = nullptr;  // [2^w], grouped by popcount
  int* d_koff = nullptr;             // [w+2]
  TileLL* d_ll = nullptr;
  TileHH* d_hh = nullptr;
  TileMX* d_mx = nullptr;
  TileMXLow* d_mxlow = nullptr;
  size_t smem_bytes = 0;
  int ctas_per_sm = 1;
};

namespace {

struct TileParams {
  int N, K, w, nh, mode;
  int n_ll, n_hh, n_mx, n_mxlow, max_run;
  uint32_t n_H;
  int64_t dim;
  const uint64_t* binom;             // [(N+1)*(K+1)]
  const uint16_t* lr_tab;
  const uint16_t* low_states;
  const int* koff;
  const TileLL* ll;
  const TileHH* hh;
  const TileMX* mx;
  const TileMXLow* mxlow;
  const uint2* clt;
  double diag0;
  ChainState* st;
  double* partials;
  unsigned int* ticket;
  int stride;
};

// base(H): number of sector labels below H << w  =  sum over set bits p of H of
// C(p + w, k + c_p), k = N_up - popc(H), c_p = set bits of H at positions <= p.
__device__ __forceinline__ uint64_t tile_base(uint32_t H, int w, int K, const uint64_t* __restrict__ binom) {
  const int K1 = K + 1;
  int c = K - __popc(H);               // ones in the low part
  uint64_t r = 0;
  uint32_t x = H;
  while (x) {
    const int p = __ffs((int)x) - 1;
    x &= x - 1;
    ++c;
    r += binom[(p + w) * K1 + c];
  }
  return r;
}

template <typename R>
struct SmemLayout {
  uint64_t* binom;       // (N+1)*(K+1)
  uint16_t* lr_tab;      // 2^w            (CR)
  uint2* clt_own;        // 2^(w-5)        (CLT)
  uint2* clt_nb;         // 2^(w-5)        (CLT)
  R* vs0;                // max_run
  R* vbuf;               // max_run
  R* acc;                // max_run
  uint16_t* Ls;          // max_run
  uint32_t* ll_mask;     // n_ll
  R* ll_J;               // n_ll
  TileHH* hh;
  TileMX* mx;
  int* mxlow_bit;        // n_mxlow
  R* mxlow_J;            // n_mxlow
  uint64_t* hh_base;     // n_hh : base of the neighbour run of each ACTIVE hh bond (compacted)
  R* hh_J;               // n_hh : its J/2
  uint64_t* mx_base;     // n_mx
  int* mx_len;           // n_mx  (0 = inactive for this run)
  int* mx_k;             // n_mx
};

template <typename R>
__host__ __device__ inline size_t tile_layout(SmemLayout<R>& s, unsigned char* p0, int N, int K, int w, int mode,
                                              int max_run, int n_ll, int n_hh, int n_mx, int n_mxlow) {
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return p0 + at; };
  s.binom = (uint64_t*)take((size_t)(N + 1) * (K + 1) * 8);
  if (mode == FTLM_INDEX_CR) { s.lr_tab = (uint16_t*)take(((size_t)1 << w) * 2); s.clt_own = nullptr; s.clt_nb = nullptr; }
  else { s.lr_tab = nullptr; s.clt_own = (uint2*)take(((size_t)1 << (w - 5)) * 8); s.clt_nb = (uint2*)take(((size_t)1 << (w - 5)) * 8); }
  s.vs0 = (R*)take((size_t)max_run * sizeof(R));
  s.vbuf = (R*)take((size_t)max_run * sizeof(R));
  s.acc = (R*)take((size_t)max_run * sizeof(R));
  s.Ls = (uint16_t*)take((size_t)max_run * 2);
  s.ll_mask = (uint32_t*)take((size_t)(n_ll ? n_ll : 1) * 4);
  s.ll_J = (R*)take((size_t)(n_ll ? n_ll : 1) * sizeof(R));
  s.hh = (TileHH*)take((size_t)(n_hh ? n_hh : 1) * sizeof(TileHH));
  s.mx = (TileMX*)take((size_t)(n_mx ? n_mx : 1) * sizeof(TileMX));
  s.mxlow_bit = (int*)take((size_t)(n_mxlow ? n_mxlow : 1) * 4);
  s.mxlow_J = (R*)take((size_t)(n_mxlow ? n_mxlow : 1) * sizeof(R));
  s.hh_base = (uint64_t*)take((size_t)(n_hh ? n_hh : 1) * 8);
  s.hh_J = (R*)take((size_t)(n_hh ? n_hh : 1) * sizeof(R));
  s.mx_base = (uint64_t*)take((size_t)(n_mx ? n_mx : 1) * 8);
  s.mx_len = (int*)take((size_t)(n_mx ? n_mx : 1) * 4);
  s.mx_k = (int*)take((size_t)(n_mx ? n_mx : 1) * 4);
  return o;
}

// local index of low word Lp inside its run, CR: chunk table; CLT: Alg. 2 on the staged chunk
template <int MODE>
__device__ __forceinline__ uint32_t local_index(uint32_t Lp, const uint16_t* __restrict__ lr_tab,
                                                const uint2* __restrict__ chunk, uint32_t chunk_base) {
  if (MODE == FTLM_INDEX_CR) return lr_tab[Lp];
  const uint2 e = chunk[Lp >> 5];
  return e.y + __popc(e.x & ((1u << (Lp & 31u)) - 1u)) - chunk_base;
}

template <typename R, int MODE, bool FUSED>
__global__ void __launch_bounds__(TILE_THREADS)
hv_tile_kernel(TileParams p, const R* __restrict__ v, const R* __restrict__ qprev, R* __restrict__ y) {
  FTLM_DYN_SMEM(smem);
  __shared__ double sh_red[96];
  __shared__ int s_nhh_active;
  __shared__ uint64_t s_base;
  if (FUSED) { if (p.st->done) return; }
  SmemLayout<R> S;
  tile_layout<R>(S, smem, p.N, p.K, p.w, MODE, p.max_run, p.n_ll, p.n_hh, p.n_mx, p.n_mxlow);
  const int tid = threadIdx.x;
  // ---- one-time staging of the tables -----------------------------------------------------
  for (int k = tid; k < (p.N + 1) * (p.K + 1); k += TILE_THREADS) S.binom[k] = p.binom[k];
  if (MODE == FTLM_INDEX_CR) {
    const uint32_t* src = (const uint32_t*)p.lr_tab;
    uint32_t* dst = (uint32_t*)S.lr_tab;
    for (int k = tid; k < (1 << (p.w - 1)); k += TILE_THREADS) dst[k] = src[k];
  }
  for (int k = tid; k < p.n_ll; k += TILE_THREADS) { S.ll_mask[k] = p.ll[k].mask; S.ll_J[k] = (R)p.ll[k].Jh; }
  for (int k = tid; k < p.n_hh; k += TILE_THREADS) S.hh[k] = p.hh[k];
  for (int k = tid; k < p.n_mx; k += TILE_THREADS) S.mx[k] = p.mx[k];
  for (int k = tid; k < p.n_mxlow; k += TILE_THREADS) { S.mxlow_bit[k] = p.mxlow[k].bit; S.mxlow_J[k] = (R)p.mxlow[k].Jh; }
  __syncthreads();

  const R bprev = FUSED ? (R)p.st->beta_prev : (R)0;
  const R diag0 = (R)p.diag0;
  const int nchunk = 1 << (p.w - 5);
  double s_qy = 0.0, s_yy = 0.0, s_qq = 0.0;

  for (uint32_t H = blockIdx.x; H < p.n_H; H += gridDim.x) {
    const int k = p.K - __popc(H);
    if (k < 0 || k > p.w) continue;                                   // no rows with this high part
    const int koff = p.koff[k];
    const int run_len = p.koff[k + 1] - koff;
    // ---- P0: CTA-uniform data of this run -------------------------------------------------
    if (tid == 0) s_base = tile_base(H, p.w, p.K, S.binom);
    if (tid >= 32 && tid < 64) {                                      // warp 1: compact active hh bonds
      const int lane = tid - 32;
      int count = 0;
      for (int b0 = 0; b0 < p.n_hh; b0 += 32) {
        const int b = b0 + lane;
        bool act = false;
        uint32_t m = 0;
        if (b < p.n_hh) { m = S.hh[b].mask; const uint32_t x = H & m; act = (x != 0 && x != m); }
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (act) {
          const int pos = count + __popc(bal & ((1u << lane) - 1u));
          S.hh_base[pos] = tile_base(H ^ m, p.w, p.K, S.binom);
          S.hh_J[pos] = (R)S.hh[b].Jh;
        }
        count += __popc(bal);
      }
      if (lane == 0) s_nhh_active = count;
    }
    if (tid >= 64 && tid < 64 + p.n_mx) {                             // mixed sites: neighbour run
      const int s = tid - 64;
      const uint32_t bit = 1u << S.mx[s].site;
      const int kp = (H & bit) ? k + 1 : k - 1;                       // low part gains / loses a one
      int len = 0;
      if (kp >= 0 && kp <= p.w) {
        len = p.koff[kp + 1] - p.koff[kp];
        S.mx_base[s] = tile_base(H ^ bit, p.w, p.K, S.binom);
      }
      S.mx_len[s] = len;
      S.mx_k[s] = kp;
    }
    __syncthreads();
    const uint64_t base = s_base;
    // ---- P1: stage the own run (and its CLT chunk) -------------------------------------------
    for (int lr = tid; lr < run_len; lr += TILE_THREADS) {
      S.vs0[lr] = v[base + lr];
      S.Ls[lr] = __ldg(&p.low_states[koff + lr]);
    }
    uint32_t own_cbase = 0;
    if (MODE == FTLM_INDEX_CLT) {
      const uint2* g = p.clt + ((size_t)H << (p.w - 5));
      for (int c = tid; c < nchunk; c += TILE_THREADS) S.clt_own[c] = __ldg(&g[c]);
      own_cbase = (uint32_t)base;
    }
    __syncthreads();
    // ---- P2: ll bonds (smem gathers) + active hh bonds (coalesced streams) --------------------
    const int nhh = s_nhh_active;
    for (int lr = tid; lr < run_len; lr += TILE_THREADS) {
      const uint32_t L = S.Ls[lr];
      const R vt = S.vs0[lr];
      R acc = 0;
      for (int b = 0; b < nhh; ++b) acc += S.hh_J[b] * (__ldg(&v[S.hh_base[b] + lr]) - vt);
      for (int b = 0; b < p.n_ll; ++b) {
        const uint32_t m = S.ll_mask[b];
        if (__popc(L & m) == 1) acc += S.ll_J[b] * (S.vs0[local_index<MODE>(L ^ m, S.lr_tab, S.clt_own, own_cbase)] - vt);
      }
      S.acc[lr] = acc;
    }
    // ---- P4: mixed bonds, one neighbour run (high site) at a time ------------------------------
    for (int s = 0; s < p.n_mx; ++s) {
      const int len = S.mx_len[s];
      if (len == 0) continue;                                         // uniform
      const uint64_t nb_base = S.mx_base[s];
      __syncthreads();                                                // vbuf (and clt_nb) free
      for (int e = tid; e < len; e += TILE_THREADS) S.vbuf[e] = __ldg(&v[nb_base + e]);
      if (MODE == FTLM_INDEX_CLT) {
        const uint2* g = p.clt + ((size_t)(H ^ (1u << S.mx[s].site)) << (p.w - 5));
        for (int c = tid; c < nchunk; c += TILE_THREADS) S.clt_nb[c] = __ldg(&g[c]);
      }
      __syncthreads();
      const uint32_t hb = (H >> S.mx[s].site) & 1u;
      const int first = S.mx[s].first, cnt = S.mx[s].count;
      for (int lr = tid; lr < run_len; lr += TILE_THREADS) {
        const uint32_t L = S.Ls[lr];
        const R vt = S.vs0[lr];
        R a = 0;
        for (int e = 0; e < cnt; ++e) {
          const int bit = S.mxlow_bit[first + e];
          if (((L >> bit) & 1u) != hb)
            a += S.mxlow_J[first + e] *
                 (S.vbuf[local_index<MODE>(L ^ (1u << bit), S.lr_tab, S.clt_nb, (uint32_t)nb_base)] - vt);
        }
        S.acc[lr] += a;
      }
    }
    // ---- P5: epilogue: diagonal, Lanczos recurrence, reductions ------------------------------
    for (int lr = tid; lr < run_len; lr += TILE_THREADS) {
      const R vt = S.vs0[lr];
      R out = diag0 * vt + S.acc[lr];
      if (FUSED) {
        out -= bprev * __ldcs(&qprev[base + lr]);
        s_qy += (double)vt * (double)out;
        s_yy += (double)out * (double)out;
        s_qq += (double)vt * (double)vt;
      }
      __stcs(&y[base + lr], out);
    }
    __syncthreads();                                                  // smem reused by the next run
  }
  if (FUSED) lanczos_finish(s_qy, s_yy, s_qq, p.partials, p.stride, p.ticket, p.st, sh_red);
}

// Neighbour indices through the TILE index path (base(H') + lr) for the bit-exact test hook.
// Thread per row; the row's own (H, L) comes from a full unrank and is cross-checked against the
// run tables (a mismatch writes -2).
template <int MODE>
__global__ void __launch_bounds__(256)
neighbors_tile_kernel(TileParams p, const BondDev* __restrict__ bonds, int nb, int64_t row0, int64_t nrows,
                      int64_t* __restrict__ out) {
  const int K1 = p.K + 1;
  for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < nrows; r += (int64_t)gridDim.x * blockDim.x) {
    const uint64_t t = (uint64_t)(row0 + r);
    uint64_t n = 0, rem = t;
    int A = p.K;
    for (int q = p.N - 1; q >= 0 && A > 0; --q) {
      const uint64_t c = p.binom[q * K1 + A];
      if (rem >= c) { n |= 1ull << q; rem -= c; --A; }
    }
    const uint32_t H = (uint32_t)(n >> p.w), L = (uint32_t)(n & ((1ull << p.w) - 1));
    const int k = __popc(L);
    const uint64_t base = tile_base(H, p.w, p.K, p.binom);
    const bool ok = (base + p.lr_tab[L] == t) && (p.low_states[p.koff[k] + p.lr_tab[L]] == L);
    for (int b = 0; b < nb; ++b) {
      const uint64_t m = bonds[b].mask, x = n & m;
      int64_t idx = -1;
      if (x != 0 && x != m) {
        const uint64_t np_ = n ^ m;
        if (MODE == FTLM_INDEX_CLT) {
          const uint2 e = p.clt[np_ >> 5];
          idx = (int64_t)e.y + __popc(e.x & ((1u << ((uint32_t)np_ & 31u)) - 1u));
        } else {
          const uint32_t Hp = (uint32_t)(np_ >> p.w), Lp = (uint32_t)(np_ & ((1ull << p.w) - 1));
          idx = (int64_t)(tile_base(Hp, p.w, p.K, p.binom) + p.lr_tab[Lp]);
        }
        if (!ok) idx = -2;
      }
      out[r * nb + b] = idx;
    }
  }
}

TileParams make_tile_params(ftlm_ctx* c) {
  TilePlan* t = c->tile;
  TileParams p;
  p.N = c->N; p.K = c->N_up; p.w = t->w; p.nh = t->nh; p.mode = c->mode;
  p.n_ll = t->n_ll; p.n_hh = t->n_hh; p.n_mx = t->n_mx; p.n_mxlow = t->n_mxlow; p.max_run = t->max_run;
  p.n_H = t->n_H; p.dim = c->dim; p.binom = c->d_binom64; p.lr_tab = t->d_lr_tab; p.low_states = t->d_low_states;
  p.koff = t->d_koff; p.ll = t->d_ll; p.hh = t->d_hh; p.mx = t->d_mx; p.mxlow = t->d_mxlow; p.clt = c->d_clt;
  p.diag0 = c->diag0; p.st = c->d_state; p.partials = c->d_partials; p.ticket = c->d_ticket; p.stride = c->max_blocks;
  return p;
}

template <typename R>
size_t tile_smem_bytes(const ftlm_ctx* c, int w, int max_run, int n_ll, int n_hh, int n_mx, int n_mxlow) {
  SmemLayout<R> S;
  return tile_layout<R>(S, nullptr, c->N, c->N_up, w, c->mode, max_run, n_ll, n_hh, n_mx, n_mxlow);
}

uint64_t binom_h(int n, int k) {
  if (k < 0 || k > n) return 0;
  if (k > n - k) k = n - k;
  unsigned __int128 r = 1;
  for (int i = 1; i <= k; ++i) r = r * (unsigned)(n - k + i) / (unsigned)i;
  return (uint64_t)r;
}

template <typename R, int MODE>
int launch_tile(ftlm_ctx* c, const TileParams& p, const void* v, const void* qp, void* y, int fused, cudaStream_t s) {
  TilePlan* t = c->tile;
  auto grid_of = [&](int per_sm) {
    int grid = c->sm_count * per_sm;
    if ((uint32_t)grid > t->n_H) grid = (int)t->n_H;
    if (grid > c->max_blocks) grid = c->max_blocks;
    return grid;
  };
  if (fused) {
    auto k = hv_tile_kernel<R, MODE, true>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t->smem_bytes));
    int occ = 1;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, TILE_THREADS, t->smem_bytes));
    FTLM_LAUNCH(k, grid_of(occ < 1 ? 1 : occ), TILE_THREADS, t->smem_bytes, s, p, (const R*)v, (const R*)qp, (R*)y);
  } else {
    auto k = hv_tile_kernel<R, MODE, false>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t->smem_bytes));
    int occ = 1;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, TILE_THREADS, t->smem_bytes));
    FTLM_LAUNCH(k, grid_of(occ < 1 ? 1 : occ), TILE_THREADS, t->smem_bytes, s, p, (const R*)v, (const R*)qp, (R*)y);
  }
  CK(cudaGetLastError());
  return FTLM_OK;
}

}  // namespace

void ftlm_tile_plan_destroy(ftlm_ctx* c) {
  TilePlan* t = c->tile;
  if (!t) return;
  cudaFree(t->d_lr_tab); cudaFree(t->d_low_states); cudaFree(t->d_koff);
  cudaFree(t->d_ll); cudaFree(t->d_hh); cudaFree(t->d_mx); cudaFree(t->d_mxlow);
  delete t;
  c->tile = nullptr;
}

// Build the plan.  Returns FTLM_OK with c->tile == nullptr when the sector is too small or the
// split is impossible (the dispatcher then uses the ROW kernels).
int ftlm_tile_plan_create(ftlm_ctx* c) {
  c->tile = nullptr;
  const int N = c->N;
  if (N < 9 || c->dim < 64) return FTLM_OK;
  const size_t smem_cap = 227 * 1024 - 1024;
  auto need = [&](int w, int nll, int nhh, int nmx, int nmxl) {
    const int mr = (int)binom_h(w, w / 2);
    return c->prec == FTLM_FP32 ? tile_smem_bytes<float>(c, w, mr, nll, nhh, nmx, nmxl)
                                : tile_smem_bytes<double>(c, w, mr, nll, nhh, nmx, nmxl);
  };
  int w = c->low_bits;
  if (w == 0) {
    // default: the largest w <= 14 that leaves >= 2 CTAs per SM; measured choice, see DESIGN.md
    w = 14;
    if (w > N - 3) w = N - 3;
    while (w > 8 && need(w, c->nb, c->nb, 32, c->nb) > smem_cap / 2) --w;
  }
  if (w < 6 || w > 16 || w > N - 1 || N - w > 31) {
    if (c->low_bits) { ftlm_set_error("low_bits=%d unusable for N=%d (need 6 <= w <= 16, N-w <= 31)", w, N); return FTLM_EINVAL; }
    return FTLM_OK;
  }
  std::vector<TileLL> ll;
  std::vector<TileHH> hh;
  std::vector<std::vector<TileMXLow>> per_site((size_t)(N - w));
  for (const BondDev& b : c->bonds) {
    if (b.j < w) { TileLL e; e.mask = (uint32_t)b.mask; e.pad = 0; e.Jh = b.Jh; ll.push_back(e); }
    else if (b.i >= w) { TileHH e; e.mask = (uint32_t)(b.mask >> w); e.pad = 0; e.Jh = b.Jh; hh.push_back(e); }
    else { TileMXLow e; e.bit = b.i; e.pad = 0; e.Jh = b.Jh; per_site[(size_t)(b.j - w)].push_back(e); }
  }
  std::vector<TileMX> mx;
  std::vector<TileMXLow> mxlow;
  for (int s = 0; s < N - w; ++s)
    if (!per_site[(size_t)s].empty()) {
      TileMX e; e.site = s; e.first = (int)mxlow.size(); e.count = (int)per_site[(size_t)s].size(); e.pad = 0;
      mx.push_back(e);
      for (auto& x : per_site[(size_t)s]) mxlow.push_back(x);
    }
  if ((int)hh.size() > TILE_MAX_HH || (int)mx.size() > TILE_MAX_SITES) {
    if (c->low_bits) { ftlm_set_error("TILE: too many hh bonds / mixed sites"); return FTLM_EUNSUPPORTED; }
    return FTLM_OK;
  }
  const size_t smem = need(w, (int)ll.size(), (int)hh.size(), (int)mx.size(), (int)mxlow.size());
  if (smem > smem_cap) {
    if (c->low_bits) { ftlm_set_error("TILE: low_bits=%d needs %zu bytes of shared memory", w, smem); return FTLM_EUNSUPPORTED; }
    return FTLM_OK;
  }
  TilePlan* t = new TilePlan();
  t->w = w; t->nh = N - w; t->n_H = 1u << (N - w);
  t->n_ll = (int)ll.size(); t->n_hh = (int)hh.size(); t->n_mx = (int)mx.size(); t->n_mxlow = (int)mxlow.size();
  t->max_run = (int)binom_h(w, w / 2);
  t->smem_bytes = smem;
  t->ctas_per_sm = (int)std::max<size_t>(1, std::min<size_t>(4, (228 * 1024) / (smem + 1024)));
  // chunk tables generated from binomials: lr(L) = sum_{p in L} C(p, c_p); states grouped by popcount
  const size_t nl = (size_t)1 << w;
  std::vector<uint16_t> lr(nl), states(nl);
  std::vector<int> koff((size_t)w + 2, 0);
  for (int k = 0; k <= w; ++k) koff[(size_t)k + 1] = koff[(size_t)k] + (int)binom_h(w, k);
  for (size_t L = 0; L < nl; ++L) {
    uint64_t r = 0;
    int cnt = 0;
    for (int p = 0; p < w; ++p)
      if ((L >> p) & 1) { ++cnt; r += binom_h(p, cnt); }
    lr[L] = (uint16_t)r;
    states[(size_t)koff[(size_t)cnt] + r] = (uint16_t)L;
  }
  c->tile = t;
  auto up = [&](void** d, const void* h, size_t bytes) -> bool {
    if (cudaMalloc(d, bytes ? bytes : 16) != cudaSuccess) return false;
    if (bytes && cudaMemcpy(*d, h, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return false;
    return true;
  };
  bool ok = up((void**)&t->d_lr_tab, lr.data(), nl * 2) && up((void**)&t->d_low_states, states.data(), nl * 2) &&
            up((void**)&t->d_koff, koff.data(), koff.size() * 4) && up((void**)&t->d_ll, ll.data(), ll.size() * sizeof(TileLL)) &&
            up((void**)&t->d_hh, hh.data(), hh.size() * sizeof(TileHH)) && up((void**)&t->d_mx, mx.data(), mx.size() * sizeof(TileMX)) &&
            up((void**)&t->d_mxlow, mxlow.data(), mxlow.size() * sizeof(TileMXLow));
  if (!ok) { cudaGetLastError(); ftlm_tile_plan_destroy(c); ftlm_set_error("TILE: table upload failed"); return FTLM_ENOMEM; }
  return FTLM_OK;
}

int ftlm_launch_hv_tile(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, cudaStream_t s) {
  if (!c->tile) { ftlm_set_error("TILE kernel unavailable"); return FTLM_EUNSUPPORTED; }
  TileParams p = make_tile_params(c);
  if (c->prec == FTLM_FP32) {
    if (c->mode == FTLM_INDEX_CLT) return launch_tile<float, FTLM_INDEX_CLT>(c, p, v, qprev, y, fused, s);
    return launch_tile<float, FTLM_INDEX_CR>(c, p, v, qprev, y, fused, s);
  }
  if (c->mode == FTLM_INDEX_CLT) return launch_tile<double, FTLM_INDEX_CLT>(c, p, v, qprev, y, fused, s);
  return launch_tile<double, FTLM_INDEX_CR>(c, p, v, qprev, y, fused, s);
}

int ftlm_launch_neighbors_tile(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s) {
  if (!c->tile) { ftlm_set_error("TILE kernel unavailable"); return FTLM_EUNSUPPORTED; }
  TileParams p = make_tile_params(c);
  int64_t blocks = (nrows + 255) / 256;
  if (blocks > c->sm_count * 8) blocks = c->sm_count * 8;
  if (c->mode == FTLM_INDEX_CLT) { auto k__ = neighbors_tile_kernel<FTLM_INDEX_CLT>; FTLM_LAUNCH(k__, (int)blocks, 256, 0, s, p, c->d_bonds, c->nb, row0, nrows, d_idx); }
  else { auto k__ = neighbors_tile_kernel<FTLM_INDEX_CR>; FTLM_LAUNCH(k__, (int)blocks, 256, 0, s, p, c->d_bonds, c->nb, row0, nrows, d_idx); }
  CK(cudaGetLastError());
  return FTLM_OK;
}
