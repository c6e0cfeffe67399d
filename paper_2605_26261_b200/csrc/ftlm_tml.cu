// TML kernels - the three-level tile of the gather H.v.
//
// A label is split n = (T << (m+w)) | (M << w) | L  (top t bits, middle m bits, low w bits).
// All rows sharing T are one contiguous "tile" of the vector (C(m+w, kT) rows, kT = N_up -
// popc(T)); inside it the rows sharing M are one contiguous "column" (C(w, kL) rows, kL = kT -
// popc(M)), ordered by lr(L) = rank of L among the w-bit words of equal popcount:
//     index(n) = base(T) + coloff[kT][M] + lr(L).
// One CTA stages one tile in shared memory; one warp owns 32 consecutive rows of one column, so
// everything that depends on (T, M) alone is warp-uniform.  The 6 bond classes (by where the two
// sites sit) cost, per row:
//   LL  in-column permutation      -> shared-memory table LLtab[bond][L] (self if parallel)
//   MM  column -> column, same lr  -> conflict-free shared-memory read, warp-uniform test
//   ML  column change + flip of L_i-> shared-memory read at FLtab[i][L], per-lane test
//   TT  tile -> tile, same offset  -> coalesced global stream (L2), tile-uniform test
//   TM  tile and column change     -> coalesced global read, warp-uniform test
//   TL  tile change + flip of L_i  -> global gather at FLtab[i][L], per-lane test
// Every bond contributes (J_b/2) (v[swap_b n] - v[n]) on top of diag0 * v[n] (Eq. 12 with the
// s=1/2 coefficients of Eqs. 13-14: an antiparallel bond has the off-diagonal element J/2 and
// lowers the diagonal from +J/4 to -J/4).
// Index strategies (bit-exact with ROW and the oracle): CR ranks T' with the binomial table in
// shared memory (Eq. 15-16 at d=2) - the rank is updated only across the flipped positions
// because coloff/FLtab/LLtab hold the low-part ranks; CLT reads base(T') = C_b of block
// (T' << (m+w)) >> 5 from the compressed table (Alg. 2 with j = 0).
// Tiles are handed out in ascending T by an atomic counter so that co-resident CTAs work on
// neighbouring tiles and flips of low T bits hit L2; per-tile FP64 partial sums are written to a
// buffer indexed by T and added in fixed order by the last CTA (bit-reproducible alpha, beta).
#include <algorithm>
#include <cstring>
#include <vector>

#include "ftlm_common.cuh"

#define TML_MAX_LL 32
#define TML_MAX_MM 32
#define TML_MAX_ML 32
#define TML_MAX_TT 64
#define TML_MAX_TS 32
#define TML_MAX_TX 64
#define TML_MAX_THREADS 1024

template <typename R>
struct TmlParams {
  int N, K, w, m, t, mw, mode;
  uint32_t nT;
  int n_ll4, n_mm, n_ml, n_tt, n_ts;
  int max_tile;
  int64_t dim;
  const uint64_t* binom;              // [(N+1)*(K+1)] global
  const uint2* clt;                   // CLT mode: base(T') = clt[T' << (mw-5)].y
  const unsigned char* blob;          // tables staged into shared memory
  int blob_bytes, off_koff, off_lstate, off_coloff, off_ll, off_fl, off_tlen;
  const uint32_t* items;              // (M | chunk << 16), grouped by kT
  const int* item_off;                // [mw + 2]
  double* partials;                   // [3][nT]
  unsigned int* counter;              // [0] tile counter, [1] ticket
  ChainState* st;
  R diag_coef;                        // diag0 - sum_{LL} J_b/2  (LL bonds are in swap form)
  R ll_J[TML_MAX_LL];
  uint32_t mm_mask[TML_MAX_MM]; R mm_J[TML_MAX_MM];
  uint8_t ml_i[TML_MAX_ML], ml_j[TML_MAX_ML]; R ml_J[TML_MAX_ML];
  uint32_t tt_mask[TML_MAX_TT]; R tt_J[TML_MAX_TT];
  uint8_t ts_site[TML_MAX_TS], ts_first[TML_MAX_TS + 1];
  uint8_t tx_kind[TML_MAX_TX], tx_i[TML_MAX_TX]; R tx_J[TML_MAX_TX];
};

struct TmlPlan {
  int w = 0, m = 0, t = 0;
  int n_ll = 0, n_ll4 = 0, n_mm = 0, n_ml = 0, n_tt = 0, n_ts = 0, n_tx = 0;
  int threads = 512, ctas_per_sm = 1, max_tile = 0;
  uint32_t nT = 0;
  size_t smem_bytes = 0;
  unsigned char* d_blob = nullptr;
  int blob_bytes = 0, off_koff = 0, off_lstate = 0, off_coloff = 0, off_ll = 0, off_fl = 0, off_tlen = 0;
  uint32_t* d_items = nullptr;
  int* d_item_off = nullptr;
  double* d_partials = nullptr;
  unsigned int* d_counter = nullptr;
  int* d_bond_class = nullptr;        // per original bond: class 0..5 (LL, MM, ML, TT, TM, TL)
  int* d_bond_entry = nullptr;        // index in the class list (TM/TL: index in tx list)
  int* d_bond_ts = nullptr;           // TM/TL: index of the T-site entry
  double diag_coef = 0.0;
  std::vector<double> ll_J, mm_J, ml_J, tt_J, tx_J;
  std::vector<uint32_t> mm_mask, tt_mask;
  std::vector<uint8_t> ml_i, ml_j, ts_site, ts_first, tx_kind, tx_i;
};

namespace {

// base(T): number of sector labels below T << mw (same combinatorial sum as Eq. 15-16 at d=2).
__device__ __forceinline__ uint64_t tml_base_cr(uint32_t T, int mw, int K, const uint64_t* __restrict__ binom) {
  const int K1 = K + 1;
  int c = K - __popc(T);
  uint64_t r = 0;
  uint32_t x = T;
  while (x) {
    const int p = __ffs((int)x) - 1;
    x &= x - 1;
    ++c;
    r += binom[(p + mw) * K1 + c];
  }
  return r;
}

template <int MODE>
__device__ __forceinline__ uint64_t tml_base(uint32_t T, int mw, int K, const uint64_t* __restrict__ binom,
                                             const uint2* __restrict__ clt) {
  if (MODE == FTLM_INDEX_CLT) return (uint64_t)__ldg(&clt[(size_t)T << (mw - 5)]).y;
  return tml_base_cr(T, mw, K, binom);
}

struct TmlSmem {
  uint64_t* binom;
  unsigned char* blob;
  unsigned char* vs;          // tile buffer (R[max_tile])
  long long* tt_base;         // [TML_MAX_TT] active TT bonds of the current tile (compacted)
  double* tt_J;               // [TML_MAX_TT] (stored as double, converted on use)
  long long* ts_base;         // [TML_MAX_TS]
  int* ts_kT;                 // [TML_MAX_TS]  (-1 = neighbour tile does not exist)
  double* red;                // [96]
  int* misc;                  // [0] tile index, [1] n active TT
  long long* base;            // [0] base of the current tile
};

__host__ __device__ inline size_t tml_layout(TmlSmem& s, unsigned char* p0, int N, int K, int blob_bytes,
                                             int max_tile, int esz) {
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return p0 + at; };
  s.binom = (uint64_t*)take((size_t)(N + 1) * (K + 1) * 8);
  s.blob = take((size_t)blob_bytes);
  s.vs = take((size_t)max_tile * esz + 16);
  s.tt_base = (long long*)take(TML_MAX_TT * 8);
  s.tt_J = (double*)take(TML_MAX_TT * 8);
  s.ts_base = (long long*)take(TML_MAX_TS * 8);
  s.ts_kT = (int*)take(TML_MAX_TS * 4);
  s.red = (double*)take(96 * 8);
  s.misc = (int*)take(16);
  s.base = (long long*)take(16);
  return o;
}

template <typename R, int MODE, bool FUSED>
__global__ void __launch_bounds__(TML_MAX_THREADS, 1)
hv_tml_kernel(const __grid_constant__ TmlParams<R> p, const R* __restrict__ v, const R* __restrict__ qprev,
              R* __restrict__ y) {
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ bool s_last;
  if (FUSED) { if (p.st->done) return; }
  TmlSmem S;
  tml_layout(S, smem, p.N, p.K, p.blob_bytes, p.max_tile, (int)sizeof(R));
  const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
  // ---- one-time staging of the tables --------------------------------------------------------
  for (int k = tid; k < (p.N + 1) * (p.K + 1); k += NT) S.binom[k] = p.binom[k];
  {
    const uint4* src = (const uint4*)p.blob;
    uint4* dst = (uint4*)S.blob;
    for (int k = tid; k < (p.blob_bytes >> 4); k += NT) dst[k] = __ldg(&src[k]);
  }
  const int* s_koff = (const int*)(S.blob + p.off_koff);
  const uint16_t* s_lstate = (const uint16_t*)(S.blob + p.off_lstate);
  const uint16_t* s_coloff = (const uint16_t*)(S.blob + p.off_coloff);       // [kT][M]
  const uint2* s_ll = (const uint2*)(S.blob + p.off_ll);                     // [group][Lidx] 4 x u16 byte offsets
  const uint16_t* s_fl = (const uint16_t*)(S.blob + p.off_fl);               // [i][Lidx] byte offset
  const int* s_tlen = (const int*)(S.blob + p.off_tlen);                     // [kT]
  const int nL = 1 << p.w, nM = 1 << p.m;
  const R bprev = FUSED ? (R)p.st->beta_prev : (R)0;
  const unsigned char* vsb0 = S.vs;

  for (;;) {
    __syncthreads();                                   // previous tile done: smem reusable
    if (tid == 0) S.misc[0] = (int)atomicAdd(&p.counter[0], 1u);
    __syncthreads();
    const uint32_t T = (uint32_t)S.misc[0];
    if (T >= p.nT) break;
    const int kT = p.K - __popc(T);
    if (kT < 0 || kT > p.mw) continue;                  // no rows with this top part
    // ---- per-tile uniform data ----------------------------------------------------------------
    if (tid == 0) S.base[0] = (long long)tml_base<MODE>(T, p.mw, p.K, S.binom, p.clt);
    if (warp == 1) {                                    // compact the active TT bonds
      int count = 0;
      for (int b0 = 0; b0 < p.n_tt; b0 += 32) {
        const int b = b0 + lane;
        bool act = false;
        uint32_t mk = 0;
        if (b < p.n_tt) { mk = p.tt_mask[b]; const uint32_t x = T & mk; act = (x != 0 && x != mk); }
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (act) {
          const int pos = count + __popc(bal & ((1u << lane) - 1u));
          S.tt_base[pos] = (long long)tml_base<MODE>(T ^ mk, p.mw, p.K, S.binom, p.clt);
          S.tt_J[pos] = (double)p.tt_J[b];
        }
        count += __popc(bal);
      }
      if (lane == 0) S.misc[1] = count;
    }
    if (warp == 2 && lane < p.n_ts) {                   // neighbour tiles of the mixed T sites
      const uint32_t bit = 1u << p.ts_site[lane];
      const int kTp = (T & bit) ? kT + 1 : kT - 1;
      const bool ok = (kTp >= 0 && kTp <= p.mw);
      S.ts_kT[lane] = ok ? kTp : -1;
      S.ts_base[lane] = ok ? (long long)tml_base<MODE>(T ^ bit, p.mw, p.K, S.binom, p.clt) : 0;
    }
    __syncthreads();
    const long long base = S.base[0];
    const int tlen = s_tlen[kT];
    // ---- stage the tile --------------------------------------------------------------------------
    {
      R* vs = (R*)S.vs;
      const R* src = v + base;
      for (int x = tid; x < tlen; x += NT) vs[x] = src[x];
    }
    __syncthreads();
    // ---- rows: one warp per (column, 32-row chunk) -------------------------------------------------
    const int it0 = p.item_off[kT], it1 = p.item_off[kT + 1];
    const int ntt = S.misc[1];
    const uint16_t* co = s_coloff + kT * nM;
    double s_qy = 0.0, s_yy = 0.0, s_qq = 0.0;
    for (int it = it0 + warp; it < it1; it += NW) {
      const uint32_t item = __ldg(&p.items[it]);
      const uint32_t M = item & 0xffffu;
      const int kL = kT - __popc(M);
      const int k0 = s_koff[kL];
      const int len = s_koff[kL + 1] - k0;
      const int lr = (int)(item >> 16) * 32 + lane;
      const bool valid = lr < len;
      const int lrc = valid ? lr : 0;
      const int Lidx = k0 + lrc;
      const int cb = co[M];
      const unsigned char* vsb = vsb0 + (size_t)cb * sizeof(R);            // column base (bytes)
      const R own = *(const R*)(vsb + (size_t)lrc * sizeof(R));
      const uint32_t Lw = s_lstate[Lidx];
      R acc = 0;
      // LL: swap form, 4 bonds per 8-byte table entry
      for (int g = 0; g < (p.n_ll4 >> 2); ++g) {
        const uint2 q = s_ll[g * nL + Lidx];
        acc += p.ll_J[4 * g + 0] * *(const R*)(vsb + (q.x & 0xffffu));
        acc += p.ll_J[4 * g + 1] * *(const R*)(vsb + (q.x >> 16));
        acc += p.ll_J[4 * g + 2] * *(const R*)(vsb + (q.y & 0xffffu));
        acc += p.ll_J[4 * g + 3] * *(const R*)(vsb + (q.y >> 16));
      }
      // MM: other column of this tile, same lr (warp-uniform test)
      for (int b = 0; b < p.n_mm; ++b) {
        const uint32_t mk = p.mm_mask[b];
        if (__popc(M & mk) == 1) {
          const R* col = (const R*)(vsb0 + (size_t)co[M ^ mk] * sizeof(R));
          acc += p.mm_J[b] * (col[lrc] - own);
        }
      }
      // ML: column M ^ bit_j, row = L with bit i flipped (per-lane test L_i != M_j)
      for (int b = 0; b < p.n_ml; ++b) {
        const int i = p.ml_i[b], j = p.ml_j[b];
        const uint32_t u = (M >> j) & 1u;
        const unsigned char* col = vsb0 + (size_t)co[M ^ (1u << j)] * sizeof(R);
        const uint32_t nb = s_fl[i * nL + Lidx];
        if (((Lw >> i) & 1u) != u) acc += p.ml_J[b] * (*(const R*)(col + nb) - own);
      }
      // TT: same offset in another tile (tile-uniform list of active bonds)
      const long long off = (long long)cb + lrc;
      for (int a = 0; a < ntt; ++a) acc += (R)S.tt_J[a] * (__ldg(&v[S.tt_base[a] + off]) - own);
      // TM / TL: neighbour tile T ^ bit_s
      for (int s = 0; s < p.n_ts; ++s) {
        const int kTp = S.ts_kT[s];
        if (kTp < 0) continue;
        const uint32_t u = (T >> p.ts_site[s]) & 1u;
        const uint16_t* cop = s_coloff + kTp * nM;
        const R* tb = v + S.ts_base[s];
        for (int e = p.ts_first[s]; e < p.ts_first[s + 1]; ++e) {
          const int i = p.tx_i[e];
          if (p.tx_kind[e] == 0) {                       // TM: column M ^ bit_i, same lr
            if (((M >> i) & 1u) != u) acc += p.tx_J[e] * (__ldg(&tb[(int)cop[M ^ (1u << i)] + lrc]) - own);
          } else {                                       // TL: column M, row flipped at L_i
            const uint32_t nb = s_fl[i * nL + Lidx];
            const unsigned char* colg = (const unsigned char*)(tb + cop[M]);
            if (((Lw >> i) & 1u) != u) acc += p.tx_J[e] * (__ldg((const R*)(colg + nb)) - own);
          }
        }
      }
      // epilogue: diagonal, Lanczos recurrence, reductions
      R out = p.diag_coef * own + acc;
      if (valid) {
        const long long g = base + off;
        if (FUSED) {
          out -= bprev * __ldcs(&qprev[g]);
          s_qy += (double)own * (double)out;
          s_yy += (double)out * (double)out;
          s_qq += (double)own * (double)own;
        }
        __stcs(&y[g], out);
      }
    }
    if (FUSED) {                                        // deterministic per-tile partial sums
      block_sum3(s_qy, s_yy, s_qq, S.red);
      if (tid == 0) {
        p.partials[T] = s_qy;
        p.partials[(size_t)p.nT + T] = s_yy;
        p.partials[2 * (size_t)p.nT + T] = s_qq;
      }
    }
  }
  // ---- grid-wide finish: the last CTA resets the counters and (fused) advances the chain ---------
  if (tid == 0) {
    __threadfence();
    s_last = (atomicAdd(&p.counter[1], 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (tid == 0) { p.counter[0] = 0; p.counter[1] = 0; }
  if (!FUSED) return;
  double a = 0.0, b = 0.0, c = 0.0;
  for (uint32_t k = tid; k < p.nT; k += NT) {            // fixed assignment and order
    a += p.partials[k]; b += p.partials[(size_t)p.nT + k]; c += p.partials[2 * (size_t)p.nT + k];
  }
  block_sum3(a, b, c, S.red);
  if (tid == 0) {
    ChainState* st = p.st;
    const int j = st->step;
    const double alpha = c > 0.0 ? a / c : 0.0;
    double b2 = c > 0.0 ? b - a * a / c : 0.0;
    if (!(b2 > 0.0)) b2 = 0.0;
    const double beta = sqrt(b2);
    st->alpha[j] = alpha;
    st->beta[j] = beta;
    double sc = st->scale;
    sc = fmax(sc, fmax(fabs(alpha), beta));
    st->scale = sc;
    st->step = j + 1;
    st->a = alpha;
    st->inv_b = beta > 0.0 ? 1.0 / beta : 0.0;
    st->beta_prev = beta;
    if (j + 1 >= st->limit || beta <= st->tol * sc) st->done = 1;
  }
}

// Neighbour indices through the TML tables (test hook; same tables, same base()/coloff/FLtab/LLtab
// arithmetic as hv_tml_kernel, read from global memory).  The row's own (T, M, L) comes from a full
// unrank and is cross-checked against the tables (a mismatch writes -2).
template <typename R, int MODE>
__global__ void __launch_bounds__(256)
neighbors_tml_kernel(const __grid_constant__ TmlParams<R> p, const BondDev* __restrict__ bonds, int nb,
                     const int* __restrict__ bclass, const int* __restrict__ bentry, const int* __restrict__ bts,
                     int64_t row0, int64_t nrows, int64_t* __restrict__ out) {
  const int K1 = p.K + 1;
  const int* koff = (const int*)(p.blob + p.off_koff);
  const uint16_t* lstate = (const uint16_t*)(p.blob + p.off_lstate);
  const uint16_t* coloff = (const uint16_t*)(p.blob + p.off_coloff);
  const uint2* ll = (const uint2*)(p.blob + p.off_ll);
  const uint16_t* fl = (const uint16_t*)(p.blob + p.off_fl);
  const int nL = 1 << p.w, nM = 1 << p.m;
  for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < nrows; r += (int64_t)gridDim.x * blockDim.x) {
    const uint64_t tr = (uint64_t)(row0 + r);
    uint64_t n = 0, rem = tr;
    int A = p.K;
    for (int q = p.N - 1; q >= 0 && A > 0; --q) {
      const uint64_t c = p.binom[q * K1 + A];
      if (rem >= c) { n |= 1ull << q; rem -= c; --A; }
    }
    const uint32_t T = (uint32_t)(n >> p.mw), M = (uint32_t)(n >> p.w) & (uint32_t)(nM - 1), L = (uint32_t)n & (uint32_t)(nL - 1);
    const int kT = p.K - __popc(T), kL = kT - __popc(M);
    const uint64_t base = tml_base<MODE>(T, p.mw, p.K, p.binom, p.clt);
    const int cb = coloff[kT * nM + M];
    const int lr = (int)(tr - base) - cb;
    const bool ok = lr >= 0 && lr < koff[kL + 1] - koff[kL] && lstate[koff[kL] + lr] == L;
    const int Lidx = ok ? koff[kL] + lr : 0;
    for (int b = 0; b < nb; ++b) {
      const uint64_t mk = bonds[b].mask, x = n & mk;
      int64_t idx = -1;
      const int e = bentry[b];
      if (x != 0 && x != mk) {
        switch (bclass[b]) {
          case 0: {                                      // LL
            const uint2 q = ll[(e >> 2) * nL + Lidx];
            const uint32_t h = (e & 2) ? q.y : q.x;
            const uint32_t nbB = (e & 1) ? (h >> 16) : (h & 0xffffu);
            idx = (int64_t)base + cb + (int)(nbB / sizeof(R));
            break;
          }
          case 1: idx = (int64_t)base + coloff[kT * nM + (M ^ p.mm_mask[e])] + lr; break;          // MM
          case 2: idx = (int64_t)base + coloff[kT * nM + (M ^ (1u << p.ml_j[e]))] +               // ML
                        (int)(fl[p.ml_i[e] * nL + Lidx] / sizeof(R)); break;
          case 3: idx = (int64_t)tml_base<MODE>(T ^ p.tt_mask[e], p.mw, p.K, p.binom, p.clt) + cb + lr; break;  // TT
          default: {                                     // TM / TL
            const int s = bts[b];
            const uint32_t bit = 1u << p.ts_site[s];
            const int kTp = (T & bit) ? kT + 1 : kT - 1;
            const uint64_t tb = tml_base<MODE>(T ^ bit, p.mw, p.K, p.binom, p.clt);
            const int i = p.tx_i[e];
            if (p.tx_kind[e] == 0) idx = (int64_t)tb + coloff[kTp * nM + (M ^ (1u << i))] + lr;
            else idx = (int64_t)tb + coloff[kTp * nM + M] + (int)(fl[i * nL + Lidx] / sizeof(R));
          }
        }
        if (!ok) idx = -2;
      } else if (bclass[b] == 0 && ok) {                 // parallel LL bond: the table must say "self"
        const uint2 q = ll[(e >> 2) * nL + Lidx];
        const uint32_t h = (e & 2) ? q.y : q.x;
        const uint32_t nbB = (e & 1) ? (h >> 16) : (h & 0xffffu);
        if ((int)(nbB / sizeof(R)) != lr) idx = -3;
      }
      out[r * nb + b] = idx;
    }
  }
}

uint64_t binom_t(int n, int k) {
  if (k < 0 || k > n) return 0;
  if (k > n - k) k = n - k;
  unsigned __int128 r = 1;
  for (int i = 1; i <= k; ++i) r = r * (unsigned)(n - k + i) / (unsigned)i;
  return (uint64_t)r;
}

template <typename R>
void fill_params(const ftlm_ctx* c, const TmlPlan* t, TmlParams<R>& p) {
  memset(&p, 0, sizeof(p));
  p.N = c->N; p.K = c->N_up; p.w = t->w; p.m = t->m; p.t = t->t; p.mw = t->w + t->m; p.mode = c->mode;
  p.nT = t->nT; p.n_ll4 = t->n_ll4; p.n_mm = t->n_mm; p.n_ml = t->n_ml; p.n_tt = t->n_tt; p.n_ts = t->n_ts;
  p.max_tile = t->max_tile; p.dim = c->dim; p.binom = c->d_binom64; p.clt = c->d_clt; p.blob = t->d_blob;
  p.blob_bytes = t->blob_bytes; p.off_koff = t->off_koff; p.off_lstate = t->off_lstate; p.off_coloff = t->off_coloff;
  p.off_ll = t->off_ll; p.off_fl = t->off_fl; p.off_tlen = t->off_tlen; p.items = t->d_items; p.item_off = t->d_item_off;
  p.partials = t->d_partials; p.counter = t->d_counter; p.st = c->d_state; p.diag_coef = (R)t->diag_coef;
  for (int k = 0; k < t->n_ll4; ++k) p.ll_J[k] = (R)t->ll_J[(size_t)k];
  for (int k = 0; k < t->n_mm; ++k) { p.mm_mask[k] = t->mm_mask[(size_t)k]; p.mm_J[k] = (R)t->mm_J[(size_t)k]; }
  for (int k = 0; k < t->n_ml; ++k) { p.ml_i[k] = t->ml_i[(size_t)k]; p.ml_j[k] = t->ml_j[(size_t)k]; p.ml_J[k] = (R)t->ml_J[(size_t)k]; }
  for (int k = 0; k < t->n_tt; ++k) { p.tt_mask[k] = t->tt_mask[(size_t)k]; p.tt_J[k] = (R)t->tt_J[(size_t)k]; }
  for (int k = 0; k < t->n_ts; ++k) p.ts_site[k] = t->ts_site[(size_t)k];
  for (int k = 0; k <= t->n_ts; ++k) p.ts_first[k] = t->ts_first[(size_t)k];
  for (int k = 0; k < t->n_tx; ++k) { p.tx_kind[k] = t->tx_kind[(size_t)k]; p.tx_i[k] = t->tx_i[(size_t)k]; p.tx_J[k] = (R)t->tx_J[(size_t)k]; }
}

size_t tml_smem_bytes(const ftlm_ctx* c, int blob_bytes, int max_tile) {
  TmlSmem S;
  return tml_layout(S, nullptr, c->N, c->N_up, blob_bytes, max_tile, (int)ftlm_elem_size(c));
}

template <typename R, int MODE>
int launch_tml(ftlm_ctx* c, const void* v, const void* qp, void* y, int fused, cudaStream_t s) {
  TmlPlan* t = c->tml;
  TmlParams<R> p;
  fill_params<R>(c, t, p);
  int grid = c->sm_count * t->ctas_per_sm;
  if ((uint32_t)grid > t->nT) grid = (int)t->nT;
  if (fused) {
    auto k = hv_tml_kernel<R, MODE, true>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t->smem_bytes));
    k<<<grid, t->threads, t->smem_bytes, s>>>(p, (const R*)v, (const R*)qp, (R*)y);
  } else {
    auto k = hv_tml_kernel<R, MODE, false>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t->smem_bytes));
    k<<<grid, t->threads, t->smem_bytes, s>>>(p, (const R*)v, (const R*)qp, (R*)y);
  }
  CK(cudaGetLastError());
  return FTLM_OK;
}

}  // namespace

void ftlm_tml_plan_destroy(ftlm_ctx* c) {
  TmlPlan* t = c->tml;
  if (!t) return;
  cudaFree(t->d_blob); cudaFree(t->d_items); cudaFree(t->d_item_off); cudaFree(t->d_partials);
  cudaFree(t->d_counter); cudaFree(t->d_bond_class); cudaFree(t->d_bond_entry); cudaFree(t->d_bond_ts);
  delete t;
  c->tml = nullptr;
}

// Build the plan.  FTLM_OK with c->tml == nullptr when no split is possible for this sector (the
// dispatcher then uses the TILE / ROW kernels).  c->low_bits / c->mid_bits (0 = auto) choose w, m.
int ftlm_tml_plan_create(ftlm_ctx* c) {
  c->tml = nullptr;
  const int N = c->N, K = c->N_up, esz = (int)ftlm_elem_size(c);
  const bool forced = c->tml_low_bits != 0 || c->tml_mid_bits != 0;
  int w = c->tml_low_bits, m = c->tml_mid_bits;
  if (!forced) {
    int mw = N - 6 < 16 ? N - 6 : 16;
    w = mw - 2 < 9 ? mw - 2 : 9;
    m = mw - w;
  } else {
    if (w == 0) w = 9;
    if (m == 0) m = 7;
  }
  const int t = N - w - m;
  auto unusable = [&](const char* why) {
    if (forced) { ftlm_set_error("TML: low_bits=%d mid_bits=%d unusable for N=%d: %s", w, m, N, why); return (int)FTLM_EUNSUPPORTED; }
    return (int)FTLM_OK;
  };
  if (w < 5 || w > 12 || m < 1 || m > 9 || w + m > 18 || t < 1 || t > 31) return unusable("need 5<=w<=12, 1<=m<=9, w+m<=18, 1<=t<=31");
  if (c->dim < 64) return unusable("sector too small");
  const int mw = w + m;
  TmlPlan* P = new TmlPlan();
  P->w = w; P->m = m; P->t = t; P->nT = 1u << t;
  std::vector<int> bclass((size_t)c->nb, 0), bentry((size_t)c->nb, 0), bts((size_t)c->nb, 0);
  struct LLb { uint32_t mask; double Jh; };
  std::vector<LLb> ll;
  std::vector<std::vector<std::pair<int, int>>> per_site((size_t)t);   // (bond, kind) per T site
  double sumJ_ll = 0.0;
  for (int b = 0; b < c->nb; ++b) {
    const BondDev& d = c->bonds[(size_t)b];
    const int i = d.i, j = d.j;                                          // i < j
    if (j < w) { bclass[(size_t)b] = 0; bentry[(size_t)b] = (int)ll.size(); ll.push_back({(uint32_t)d.mask, d.Jh}); sumJ_ll += d.Jh; }
    else if (i >= w && j < mw) { bclass[(size_t)b] = 1; bentry[(size_t)b] = (int)P->mm_mask.size(); P->mm_mask.push_back((uint32_t)(d.mask >> w)); P->mm_J.push_back(d.Jh); }
    else if (i < w && j < mw) { bclass[(size_t)b] = 2; bentry[(size_t)b] = (int)P->ml_i.size(); P->ml_i.push_back((uint8_t)i); P->ml_j.push_back((uint8_t)(j - w)); P->ml_J.push_back(d.Jh); }
    else if (i >= mw) { bclass[(size_t)b] = 3; bentry[(size_t)b] = (int)P->tt_mask.size(); P->tt_mask.push_back((uint32_t)(d.mask >> mw)); P->tt_J.push_back(d.Jh); }
    else { bclass[(size_t)b] = i >= w ? 4 : 5; per_site[(size_t)(j - mw)].push_back({b, i >= w ? 0 : 1}); }
  }
  P->ts_first.push_back(0);
  for (int s = 0; s < t; ++s) {
    if (per_site[(size_t)s].empty()) continue;
    for (int kind = 0; kind < 2; ++kind)
      for (auto& e : per_site[(size_t)s]) {
        if (e.second != kind) continue;
        const BondDev& d = c->bonds[(size_t)e.first];
        bentry[(size_t)e.first] = (int)P->tx_kind.size();
        bts[(size_t)e.first] = (int)P->ts_site.size();
        P->tx_kind.push_back((uint8_t)kind);
        P->tx_i.push_back((uint8_t)(kind == 0 ? d.i - w : d.i));
        P->tx_J.push_back(d.Jh);
      }
    P->ts_site.push_back((uint8_t)s);
    P->ts_first.push_back((uint8_t)P->tx_kind.size());
  }
  P->n_ll = (int)ll.size(); P->n_ll4 = (P->n_ll + 3) & ~3;
  P->n_mm = (int)P->mm_mask.size(); P->n_ml = (int)P->ml_i.size(); P->n_tt = (int)P->tt_mask.size();
  P->n_ts = (int)P->ts_site.size(); P->n_tx = (int)P->tx_kind.size();
  if (P->n_ll4 > TML_MAX_LL || P->n_mm > TML_MAX_MM || P->n_ml > TML_MAX_ML || P->n_tt > TML_MAX_TT ||
      P->n_ts > TML_MAX_TS || P->n_tx > TML_MAX_TX) { delete P; return unusable("too many bonds in one class"); }
  for (int k = 0; k < P->n_ll4; ++k) P->ll_J.push_back(k < P->n_ll ? ll[(size_t)k].Jh : 0.0);
  P->diag_coef = c->diag0 - sumJ_ll;
  // ---- tables (blob) ---------------------------------------------------------------------------
  const int nL = 1 << w, nM = 1 << m;
  std::vector<int> koff((size_t)w + 2, 0);
  for (int k = 0; k <= w; ++k) koff[(size_t)k + 1] = koff[(size_t)k] + (int)binom_t(w, k);
  std::vector<uint16_t> lr((size_t)nL), lstate((size_t)nL);
  for (int L = 0; L < nL; ++L) {
    uint64_t r = 0;
    int cnt = 0;
    for (int q = 0; q < w; ++q)
      if ((L >> q) & 1) { ++cnt; r += binom_t(q, cnt); }
    lr[(size_t)L] = (uint16_t)r;
    lstate[(size_t)(koff[(size_t)cnt] + (int)r)] = (uint16_t)L;
  }
  P->max_tile = (int)binom_t(mw, mw / 2);
  if (P->max_tile > 65535 || (size_t)binom_t(w, w / 2) * (size_t)esz > 65535) { delete P; return unusable("tile too large for 16-bit offsets"); }
  std::vector<int> tlen((size_t)mw + 1);
  std::vector<uint16_t> coloff((size_t)(mw + 1) * nM, 0);
  std::vector<uint32_t> items;
  std::vector<int> item_off((size_t)mw + 2, 0);
  for (int kT = 0; kT <= mw; ++kT) {
    tlen[(size_t)kT] = (int)binom_t(mw, kT);
    int off = 0;
    for (int M = 0; M < nM; ++M) {
      coloff[(size_t)kT * nM + M] = (uint16_t)off;
      const int kL = kT - __builtin_popcount((unsigned)M);
      if (kL < 0 || kL > w) continue;
      const int len = (int)binom_t(w, kL);
      for (int ch = 0; ch * 32 < len; ++ch) items.push_back((uint32_t)M | ((uint32_t)ch << 16));
      off += len;
    }
    item_off[(size_t)kT + 1] = (int)items.size();
  }
  std::vector<uint16_t> lltab((size_t)(P->n_ll4 / 4) * nL * 4, 0), fltab((size_t)w * nL, 0);
  for (int k = 0; k <= w; ++k)
    for (int r = 0; r < koff[(size_t)k + 1] - koff[(size_t)k]; ++r) {
      const int Lidx = koff[(size_t)k] + r;
      const uint32_t L = lstate[(size_t)Lidx];
      for (int b = 0; b < P->n_ll4; ++b) {
        uint32_t nb = (uint32_t)r;                                       // self if parallel / padding
        if (b < P->n_ll) {
          const uint32_t mk = ll[(size_t)b].mask, x = L & mk;
          if (x != 0 && x != mk) nb = lr[(size_t)(L ^ mk)];
        }
        lltab[((size_t)(b >> 2) * nL + Lidx) * 4 + (b & 3)] = (uint16_t)(nb * (uint32_t)esz);
      }
      for (int i = 0; i < w; ++i) fltab[(size_t)i * nL + Lidx] = (uint16_t)((uint32_t)lr[(size_t)(L ^ (1u << i))] * (uint32_t)esz);
    }
  std::vector<unsigned char> blob;
  auto put = [&](const void* src, size_t bytes) {
    const size_t at = blob.size();
    blob.resize(at + ((bytes + 15) & ~(size_t)15), 0);
    if (bytes) memcpy(blob.data() + at, src, bytes);
    return (int)at;
  };
  P->off_koff = put(koff.data(), koff.size() * 4);
  P->off_tlen = put(tlen.data(), tlen.size() * 4);
  P->off_lstate = put(lstate.data(), lstate.size() * 2);
  P->off_coloff = put(coloff.data(), coloff.size() * 2);
  P->off_ll = put(lltab.data(), lltab.size() * 2);
  P->off_fl = put(fltab.data(), fltab.size() * 2);
  P->blob_bytes = (int)blob.size();
  P->smem_bytes = tml_smem_bytes(c, P->blob_bytes, P->max_tile);
  const size_t cap = 227 * 1024 - 1024;
  if (P->smem_bytes > cap) { delete P; return unusable("tables + tile exceed shared memory"); }
  if (P->smem_bytes + 1024 <= (228 * 1024) / 2) { P->ctas_per_sm = 2; P->threads = 512; }
  else { P->ctas_per_sm = 1; P->threads = 1024; }
  // ---- upload ----------------------------------------------------------------------------------
  c->tml = P;
  auto up = [&](void** d, const void* h, size_t bytes) -> bool {
    if (cudaMalloc(d, bytes ? bytes : 16) != cudaSuccess) return false;
    if (bytes && h && cudaMemcpy(*d, h, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return false;
    return true;
  };
  bool ok = up((void**)&P->d_blob, blob.data(), blob.size()) && up((void**)&P->d_items, items.data(), items.size() * 4) &&
            up((void**)&P->d_item_off, item_off.data(), item_off.size() * 4) &&
            up((void**)&P->d_bond_class, bclass.data(), bclass.size() * 4) &&
            up((void**)&P->d_bond_entry, bentry.data(), bentry.size() * 4) && up((void**)&P->d_bond_ts, bts.data(), bts.size() * 4) &&
            up((void**)&P->d_partials, nullptr, (size_t)P->nT * 24) && up((void**)&P->d_counter, nullptr, 16);
  if (ok) ok = cudaMemset(P->d_partials, 0, (size_t)P->nT * 24) == cudaSuccess && cudaMemset(P->d_counter, 0, 16) == cudaSuccess;
  if (!ok) { cudaGetLastError(); ftlm_tml_plan_destroy(c); ftlm_set_error("TML: table upload failed"); return FTLM_ENOMEM; }
  return FTLM_OK;
}

int64_t ftlm_tml_info(const ftlm_ctx* c, const char* key) {
  const TmlPlan* t = c->tml;
  if (!t) return -1;
  if (!strcmp(key, "tml_w")) return t->w;
  if (!strcmp(key, "tml_m")) return t->m;
  if (!strcmp(key, "tml_smem")) return (int64_t)t->smem_bytes;
  if (!strcmp(key, "tml_ctas_per_sm")) return t->ctas_per_sm;
  if (!strcmp(key, "tml_threads")) return t->threads;
  if (!strcmp(key, "tml_n_ll")) return t->n_ll;
  if (!strcmp(key, "tml_n_mm")) return t->n_mm;
  if (!strcmp(key, "tml_n_ml")) return t->n_ml;
  if (!strcmp(key, "tml_n_tt")) return t->n_tt;
  if (!strcmp(key, "tml_n_tm")) { int n = 0; for (auto k : t->tx_kind) n += (k == 0); return n; }
  if (!strcmp(key, "tml_n_tl")) { int n = 0; for (auto k : t->tx_kind) n += (k == 1); return n; }
  return -1;
}

int ftlm_launch_hv_tml(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, cudaStream_t s) {
  if (!c->tml) { ftlm_set_error("TML kernel unavailable"); return FTLM_EUNSUPPORTED; }
  if (c->prec == FTLM_FP32) {
    if (c->mode == FTLM_INDEX_CLT) return launch_tml<float, FTLM_INDEX_CLT>(c, v, qprev, y, fused, s);
    return launch_tml<float, FTLM_INDEX_CR>(c, v, qprev, y, fused, s);
  }
  if (c->mode == FTLM_INDEX_CLT) return launch_tml<double, FTLM_INDEX_CLT>(c, v, qprev, y, fused, s);
  return launch_tml<double, FTLM_INDEX_CR>(c, v, qprev, y, fused, s);
}

int ftlm_launch_neighbors_tml(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s) {
  TmlPlan* t = c->tml;
  if (!t) { ftlm_set_error("TML kernel unavailable"); return FTLM_EUNSUPPORTED; }
  int64_t blocks = (nrows + 255) / 256;
  if (blocks > c->sm_count * 8) blocks = c->sm_count * 8;
#define LAUNCHN(R, MODE)                                                                                   \
  do {                                                                                                     \
    TmlParams<R> p;                                                                                        \
    fill_params<R>(c, t, p);                                                                               \
    neighbors_tml_kernel<R, MODE><<<(int)blocks, 256, 0, s>>>(p, c->d_bonds, c->nb, t->d_bond_class,        \
                                                               t->d_bond_entry, t->d_bond_ts, row0, nrows, d_idx); \
  } while (0)
  if (c->prec == FTLM_FP32) { if (c->mode == FTLM_INDEX_CLT) LAUNCHN(float, FTLM_INDEX_CLT); else LAUNCHN(float, FTLM_INDEX_CR); }
  else { if (c->mode == FTLM_INDEX_CLT) LAUNCHN(double, FTLM_INDEX_CLT); else LAUNCHN(double, FTLM_INDEX_CR); }
#undef LAUNCHN
  CK(cudaGetLastError());
  return FTLM_OK;
}
