// TML kernels - the three-level tile of the gather H.v.
//
// A label is split n = (T << (m+w)) | (M << w) | L  (top t bits, middle m bits, low w bits).
// All rows sharing T are one contiguous "tile" of the vector (C(m+w, kT) rows, kT = N_up -
// popc(T)); inside it the rows sharing M are one contiguous "column" (C(w, kL) rows, kL = kT -
// popc(M)), ordered by lr(L) = rank of L among the w-bit words of equal popcount:
//     index(n) = base(T) + coloff[kT][M] + lr(L).
// One CTA stages one tile in shared memory; one warp owns up to 4 x 32 consecutive rows of one
// column, so everything that depends on (T, M) alone is warp-uniform.  Per column the warp first
// builds, cooperatively (lane e handles list entry e), compact descriptor lists in its own
// shared-memory scratch; the row loop then only walks those lists.  The 6 bond classes:
//   LL  in-column permutation       -> table LLtab[bond][L] in shared memory (self if parallel)
//   MM  column -> column, same lr   -> S list {column offset, J}: conflict-free smem read
//   ML  column change + flip of L_i -> FS list {column offset, J, i, M_j}: smem read at FLtab[i][L]
//   TT  tile -> tile, same offset   -> U list {row offset, J}: coalesced global read (L2)
//   TM  tile and column change      -> U list, coalesced global read
//   TL  tile change + flip of L_i   -> FG list: global gather at FLtab[i][L]
// S and U lists hold only the bonds that are antiparallel for this (T, M); the FS/FG tests
// (L_i != partner bit) are per lane.  Every bond contributes (J_b/2) (v[swap_b n] - v[n]) on top
// of diag0 * v[n] (Eq. 12 with the s=1/2 coefficients of Eqs. 13-14: an antiparallel bond has the
// off-diagonal element J/2 and lowers the diagonal from +J/4 to -J/4).
// B interleaved vectors (v[t][B]) share all of the index work (the paper's batched Lanczos,
// L207, L309).
// Index strategies (bit-exact with ROW and the oracle): CR ranks T' with the binomial table in
// shared memory (Eq. 15-16 at d=2) - the rank is updated only across the flipped positions
// because coloff/FLtab/LLtab hold the low-part ranks; CLT reads base(T') = C_b of block
// (T' << (m+w)) >> 5 from the compressed table (Alg. 2 with j = 0).
// Tiles are handed out in ascending T by an atomic counter so that co-resident CTAs work on
// neighbouring tiles and flips of low T bits hit L2; per-tile FP64 partial sums are written to a
// buffer indexed by T and added in fixed order by the last CTA (bit-reproducible alpha, beta).
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <type_traits>
#include <vector>

#define FTLM_TU 3
#include "ftlm_passb.cuh"
#include "ftlm_vec.cuh"

#define TML_MAX_LL 32
#define TML_MAX_TT 64
#define TML_MAX_TS 32
#define TML_MAX_LIST 64            // entries per static list (MM, ML, TM, TL)
#define TML_MAX_CHUNKS 8           // 32-row chunks per work item

struct TmlSEnt { uint32_t a, b; double J; };   // static list entry (see the plan builder)

template <typename R>
struct TmlParams {
  int N, K, w, m, t, mw, mode;
  uint32_t nT;
  uint32_t t_begin, t_end;            // tiles handed out: [t_begin, t_end)  (all of [0, nT) unless option "debug_items")
  int n_ll4, n_mm, n_ml, n_tt, n_ts, n_tm, n_tl;
  int max_tile, scratch_bytes;
  int64_t dim;
  const uint64_t* binom;              // [(N+1)*(K+1)] global
  const uint2* clt;                   // CLT mode: base(T') = clt[T' << (mw-5)].y
  const unsigned char* blob;          // tables staged into shared memory
  int blob_bytes, off_koff, off_tlen, off_coloff, off_ll, off_fl, off_mm, off_ml, off_tm, off_tl;
  const uint32_t* items;              // M | chunk0 << 16 | nchunks << 24, grouped by kT
  const int* item_off;                // [mw + 2]
  double* partials;                   // [3*B][nT]
  unsigned int* counter;              // [0] tile counter, [1] ticket
  ChainState* st;                     // [B]
  R diag_coef;                        // diag0 - sum_{LL} J_b/2  (LL bonds are in swap form)
  R ll_J[TML_MAX_LL];
  uint32_t tt_mask[TML_MAX_TT]; double tt_J[TML_MAX_TT];
  uint8_t ts_site[TML_MAX_TS];
  int pb_lo[8];                       // low end of PASS-B window k (neighbour test hook only)
};

struct TmlPlan {
  int w = 0, m = 0, t = 0;
  int n_ll = 0, n_ll4 = 0, n_mm = 0, n_ml = 0, n_tt = 0, n_ts = 0, n_tm = 0, n_tl = 0;
  int max_tile = 0;
  uint32_t nT = 0;
  unsigned char* d_blob = nullptr;
  int blob_bytes = 0, off_koff = 0, off_tlen = 0, off_coloff = 0, off_ll = 0, off_fl = 0, off_mm = 0, off_ml = 0,
      off_tm = 0, off_tl = 0;
  uint32_t* d_items = nullptr;
  int* d_item_off = nullptr;
  double* d_partials = nullptr;       // [3 * max_batch][nT]
  int partials_batch = 0;
  unsigned int* d_counter = nullptr;
  int* d_bond_class = nullptr;        // per original bond: class 0..5 (LL, MM, ML, TT, TM, TL)
  int* d_bond_entry = nullptr;        // index in the class list
  double diag_coef = 0.0;
  std::vector<double> ll_J, tt_J;
  std::vector<uint32_t> tt_mask;
  std::vector<uint8_t> ts_site;
  std::vector<TmlSEnt> mm, ml, tm, tl;
  std::vector<int> h_bond_class, h_bond_entry;   // host copies (option "tml_bclass:<b>")
};

namespace {

// descriptor entries of the per-warp scratch lists
template <typename R> struct UEnt;      // uniform gather: {offset, J}
template <> struct __align__(8) UEnt<float> { uint32_t off; float J; };
template <> struct __align__(16) UEnt<double> { uint32_t off, pad; double J; };
// flip gather: {row offset of the target column minus (!u << 15), J, FLtab row offset (bytes), u << 15}:
// an active lane (L_i != u) reads FLtab = row | (!u << 15), so target row = off + FLtab entry.
template <typename R> struct FEnt;
template <> struct __align__(16) FEnt<float> { uint32_t off; float J; uint32_t fl, uw; };
template <> struct __align__(16) FEnt<double> { uint32_t off, fl; double J; uint32_t uw, pad0, pad1, pad2; };
struct TmlTx { uint32_t off; int cofs; uint32_t u; int valid; };   // per-tile data of one TM / TL entry

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
    r += LD_A(&binom[(p + mw) * K1 + c]);
  }
  return r;
}

template <int MODE>
__device__ __forceinline__ uint64_t tml_base(uint32_t T, int mw, int K, const uint64_t* __restrict__ binom,
                                             const uint2* __restrict__ clt) {
  if (MODE == FTLM_INDEX_CLT) return (uint64_t)LDG(&clt[(size_t)T << (mw - 5)]).y;
  return tml_base_cr(T, mw, K, binom);
}

struct TmlSmem {
  uint64_t* binom;
  unsigned char* blob;
  unsigned char* vs;          // tile buffer (B * R [max_tile])
  uint32_t* tt_off;           // [TML_MAX_TT] base of the neighbour tile of each ACTIVE TT bond (compacted)
  double* tt_J;               // [TML_MAX_TT]
  TmlTx* txm;                 // [TML_MAX_LIST] per-tile data of the TM entries
  TmlTx* txl;                 // [TML_MAX_LIST] per-tile data of the TL entries
  double* red;                // [32 warps][3 * B]
  int* misc;                  // [0] tile index, [1] n active TT
  unsigned char* scratch;     // [warps][scratch_bytes]
};

__host__ __device__ inline size_t tml_layout(TmlSmem& s, unsigned char* p0, int N, int K, int blob_bytes,
                                             int max_tile, int row_bytes, int batch, int warps, int scratch_bytes) {
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return p0 + at; };
  s.binom = (uint64_t*)take((size_t)(N + 1) * (K + 1) * 8);
  s.blob = take((size_t)blob_bytes);
  s.vs = take((size_t)max_tile * row_bytes + 32);
  s.tt_off = (uint32_t*)take(TML_MAX_TT * 4);
  s.tt_J = (double*)take(TML_MAX_TT * 8);
  s.txm = (TmlTx*)take(TML_MAX_LIST * sizeof(TmlTx));
  s.txl = (TmlTx*)take(TML_MAX_LIST * sizeof(TmlTx));
  s.red = (double*)take((size_t)32 * 3 * batch * 8);
  s.misc = (int*)take(16);
  s.scratch = take((size_t)warps * scratch_bytes);
  return o;
}

__host__ __device__ inline int tml_scratch_bytes(int esz, int n_tt, int n_tm, int n_mm, int n_ml, int n_tl) {
  const int ue = esz == 4 ? 8 : 16, fe = esz == 4 ? 16 : 32;
  auto r16 = [](int x) { return (x + 15) & ~15; };
  return r16((n_tt + n_tm + 4) * ue) + r16((n_mm + 4) * ue) + r16((n_ml + 4) * fe) + r16((n_tl + 4) * fe);
}

__device__ __forceinline__ void load_fent(const FEnt<float>* e, uint32_t& off, float& J, uint32_t& fl, uint32_t& uw) {
  const uint4 q = LD_S((const uint4*)e);
  off = q.x; J = __uint_as_float(q.y); fl = q.z; uw = q.w;
}
__device__ __forceinline__ void load_fent(const FEnt<double>* e, uint32_t& off, double& J, uint32_t& fl, uint32_t& uw) {
  const FEnt<double> q = LD_S(e);
  off = q.off; fl = q.fl; J = q.J; uw = q.uw;
}
__device__ __forceinline__ const void* addr_u32(const void* base, uint32_t idx, uint32_t scale) {
#ifdef FTLM_EMU
  return (const void*)((const unsigned char*)base + (unsigned long long)idx * scale);
#else
  unsigned long long a;
  asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(a) : "r"(idx), "r"(scale), "l"((unsigned long long)base));
  return (const void*)a;
#endif
}

// FUSED: 0 = y = H v;  1 = fused Lanczos pass (subtract beta q_prev, FP64 sums, finish);
//        2 = first pass of a two-pass step: subtract beta q_prev only - PASS-B, which writes the final y,
//            carries the sums and the finish.
template <typename R, int B, int MODE, int FUSED>
__global__ void __launch_bounds__(B >= 4 ? 512 : 1024, 1)
hv_tml_kernel(const __grid_constant__ TmlParams<R> p, const R* __restrict__ v_, const R* __restrict__ qprev_,
              R* __restrict__ y_) {
  typedef Vec<R, B> V;
  constexpr int RB = (int)sizeof(V);                    // bytes per row
  FTLM_DYN_SMEM(smem);
  __shared__ bool s_last;
  if (FUSED) {
    bool all_done = true;
#pragma unroll
    for (int b = 0; b < B; ++b) all_done = all_done && p.st[b].done;
    if (all_done) return;
  }
  const V* __restrict__ v = (const V*)v_;
  const V* __restrict__ qprev = (const V*)qprev_;
  V* __restrict__ y = (V*)y_;
  const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
  TmlSmem S;
  tml_layout(S, smem, p.N, p.K, p.blob_bytes, p.max_tile, RB, B, NW, p.scratch_bytes);
  // ---- one-time staging of the tables --------------------------------------------------------
  for (int k = tid; k < (p.N + 1) * (p.K + 1); k += NT) ST_S(&S.binom[k], LD_G(&p.binom[k]));
  {
    const uint4* src = (const uint4*)p.blob;
    uint4* dst = (uint4*)S.blob;
    for (int k = tid; k < (p.blob_bytes >> 4); k += NT) ST_S(&dst[k], LDG(&src[k]));
  }
  const int* s_koff = (const int*)(S.blob + p.off_koff);
  const int* s_tlen = (const int*)(S.blob + p.off_tlen);
  const uint16_t* s_coloff = (const uint16_t*)(S.blob + p.off_coloff);       // [kT][M]
  const uint2* s_ll = (const uint2*)(S.blob + p.off_ll);                     // [group][Lidx] 4 x u16 rows
  const unsigned char* s_fl = S.blob + p.off_fl;                             // u16 [i][Lidx]: row | L_i << 15
  const TmlSEnt* s_mm = (const TmlSEnt*)(S.blob + p.off_mm);
  const TmlSEnt* s_ml = (const TmlSEnt*)(S.blob + p.off_ml);
  const TmlSEnt* s_tm = (const TmlSEnt*)(S.blob + p.off_tm);
  const TmlSEnt* s_tl = (const TmlSEnt*)(S.blob + p.off_tl);
  const int nL = 1 << p.w, nM = 1 << p.m;
  // per-warp scratch lists
  auto r16 = [](int x) { return (x + 15) & ~15; };
  unsigned char* sc = S.scratch + (size_t)warp * p.scratch_bytes;
  UEnt<R>* const Ul = (UEnt<R>*)sc;
  UEnt<R>* const Sl = (UEnt<R>*)(sc + r16((p.n_tt + p.n_tm + 4) * (int)sizeof(UEnt<R>)));
  FEnt<R>* const FSl = (FEnt<R>*)((unsigned char*)Sl + r16((p.n_mm + 4) * (int)sizeof(UEnt<R>)));
  FEnt<R>* const FGl = (FEnt<R>*)((unsigned char*)FSl + r16((p.n_ml + 4) * (int)sizeof(FEnt<R>)));
  V bprev;
#pragma unroll
  for (int b = 0; b < B; ++b) bprev.x[b] = FUSED ? (R)p.st[b].beta_prev : (R)0;
  const unsigned ltmask = (1u << lane) - 1u;

  for (;;) {
    __syncthreads();                                   // previous tile done: smem reusable
    if (tid == 0) S.misc[0] = (int)atomicAdd(&p.counter[0], 1u);
    __syncthreads();
    const uint32_t T = (uint32_t)S.misc[0] + p.t_begin;
    if (T >= p.t_end) break;
    const int kT = p.K - __popc(T);
    if (kT < 0 || kT > p.mw) continue;                  // no rows with this top part
    // ---- per-tile uniform data ----------------------------------------------------------------
    if (warp == 1) {                                    // compact the active TT bonds
      int count = 0;
      for (int b0 = 0; b0 < p.n_tt; b0 += 32) {
        const int b = b0 + lane;
        bool act = false;
        uint32_t mk = 0;
        if (b < p.n_tt) { mk = p.tt_mask[b]; const uint32_t x = T & mk; act = (x != 0 && x != mk); }
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (act) {
          const int pos = count + __popc(bal & ltmask);
          ST_S(&S.tt_off[pos], (uint32_t)tml_base<MODE>(T ^ mk, p.mw, p.K, S.binom, p.clt));
          ST_S(&S.tt_J[pos], p.tt_J[b]);
        }
        count += __popc(bal);
      }
      if (lane == 0) S.misc[1] = count;
    }
    if (warp == 2 || warp == 3) {                       // neighbour tile of every TM (warp 2) / TL (warp 3) entry
      const int n = warp == 2 ? p.n_tm : p.n_tl;
      const TmlSEnt* src = warp == 2 ? s_tm : s_tl;
      TmlTx* dst = warp == 2 ? S.txm : S.txl;
      for (int e = lane; e < n; e += 32) {
        const TmlSEnt d = LD_S(&src[e]);
        const uint32_t site = p.ts_site[d.b & (TML_MAX_TS - 1)], bit = 1u << site;
        const int kTp = (T & bit) ? kT + 1 : kT - 1;
        const bool ok = (kTp >= 0 && kTp <= p.mw);
        TmlTx x;
        x.off = ok ? (uint32_t)tml_base<MODE>(T ^ bit, p.mw, p.K, S.binom, p.clt) : 0u;
        x.cofs = ok ? kTp * nM : 0;
        x.u = (T >> site) & 1u;
        x.valid = ok ? 1 : 0;
        ST_S(&dst[e], x);
      }
    }
    const uint32_t base = (uint32_t)tml_base<MODE>(T, p.mw, p.K, S.binom, p.clt);
    const int tlen = LD_S(&s_tlen[kT]);
    // ---- stage the tile (16-byte loads on the aligned interior; smem keeps the global misalignment) ----
    const int mis = (RB >= 16) ? 0 : (int)(base & (uint32_t)(16 / RB - 1));   // rows past a 16-byte boundary
    const unsigned char* vsb0 = S.vs + (size_t)mis * RB;                        // row 0 of the tile
    {
      constexpr int RPV = RB >= 16 ? 1 : 16 / RB;                                // rows per 16 bytes
      const V* src = v + base;
      V* vs = (V*)vsb0;
      if (RPV == 1) {
        for (int x = tid; x < tlen; x += NT) ST_S(&vs[x], LD_G(&src[x]));
      } else {
        const int head = mis ? (RPV - mis) : 0;                                  // rows before the first boundary
        const int h = head < tlen ? head : tlen;
        const int nvec = (tlen - h) / RPV;
        if (tid < h) ST_S(&vs[tid], LD_G(&src[tid]));
        const uint4* s4 = (const uint4*)(src + h);
        uint4* d4 = (uint4*)(vs + h);
#pragma unroll 4
        for (int x = tid; x < nvec; x += NT) ST_S(&d4[x], LD_G(&s4[x]));
        const int done = h + nvec * RPV;
        if (tid < tlen - done) ST_S(&vs[done + tid], LD_G(&src[done + tid]));
      }
    }
    __syncthreads();
    // ---- rows: one warp per column (up to 8 chunks of 32 rows) ---------------------------------------
    const int it0 = LD_G(&p.item_off[kT]), it1 = LD_G(&p.item_off[kT + 1]);
    const int ntt = S.misc[1];
    const uint16_t* co = s_coloff + kT * nM;
    double s_qy[B], s_yy[B], s_qq[B];
#pragma unroll
    for (int b = 0; b < B; ++b) { s_qy[b] = 0.0; s_yy[b] = 0.0; s_qq[b] = 0.0; }
    (void)s_qy; (void)s_yy; (void)s_qq;
    for (int it = it0 + warp; it < it1; it += NW) {
      const uint32_t item = LDG(&p.items[it]);
      const uint32_t M = item & 0xffffu;
      const int chunk0 = (int)((item >> 16) & 0xffu), nch = (int)(item >> 24);
      const int kL = kT - __popc(M);
      const int k0 = LD_S(&s_koff[kL]);
      const int len = LD_S(&s_koff[kL + 1]) - k0;
      const uint32_t cb = LD_S(&co[M]);
      // ---- build the descriptor lists of this column (lane e <-> list entry e) ---------------------
      __syncwarp();
      int nU = ntt, nS = 0, nFG = 0;
      const int nFS = p.n_ml;
      R sumJ = 0;                                       // J of the uniform (U, S) entries: folded into the diagonal
      for (int a = lane; a < ntt; a += 32) {             // TT: same offset in tile T ^ mask
        const R J = (R)LD_S(&S.tt_J[a]);
        ST_S(&Ul[a].off, LD_S(&S.tt_off[a]) + cb); ST_S(&Ul[a].J, J); sumJ += J;
      }
      for (int e0 = 0; e0 < p.n_tm; e0 += 32) {          // TM: tile T ^ bit_s, column M ^ bit_i, same lr
        const int e = e0 + lane;
        bool act = false;
        uint32_t off = 0;
        R J = 0;
        if (e < p.n_tm) {
          const TmlTx x = LD_S(&S.txm[e]);
          const TmlSEnt dtm = LD_S(&s_tm[e]);
          const uint32_t i = dtm.a;
          act = x.valid && ((M >> i) & 1u) != x.u;
          if (act) { off = x.off + LD_S(&s_coloff[x.cofs + (int)(M ^ (1u << i))]); J = (R)dtm.J; }
        }
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (act) { const int pos = nU + __popc(bal & ltmask); ST_S(&Ul[pos].off, off); ST_S(&Ul[pos].J, J); sumJ += J; }
        nU += __popc(bal);
      }
      for (int e0 = 0; e0 < p.n_mm; e0 += 32) {          // MM: column M ^ mask of this tile, same lr
        const int e = e0 + lane;
        bool act = false;
        uint32_t off = 0;
        R J = 0;
        if (e < p.n_mm) {
          const TmlSEnt d = LD_S(&s_mm[e]);
          act = __popc(M & d.a) == 1;
          if (act) { off = (uint32_t)LD_S(&co[M ^ d.a]) * RB; J = (R)d.J; }
        }
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (act) { const int pos = nS + __popc(bal & ltmask); ST_S(&Sl[pos].off, off); ST_S(&Sl[pos].J, J); sumJ += J; }
        nS += __popc(bal);
      }
      for (int e = lane; e < nFS; e += 32) {             // ML: column M ^ bit_j, row flipped at L_i
        const TmlSEnt d = LD_S(&s_ml[e]);
        const uint32_t u = (M >> d.b) & 1u;
        FEnt<R> fe{};
        fe.off = (uint32_t)LD_S(&co[M ^ (1u << d.b)]) - ((u ^ 1u) << 15);
        fe.J = (R)d.J;
        fe.fl = d.a * (uint32_t)nL * 2u;
        fe.uw = u << 15;
        ST_S(&FSl[e], fe);
      }
      for (int e0 = 0; e0 < p.n_tl; e0 += 32) {          // TL: tile T ^ bit_s, column M, row flipped at L_i
        const int e = e0 + lane;
        bool act = false;
        TmlTx x;
        if (e < p.n_tl) { x = LD_S(&S.txl[e]); act = x.valid != 0; }
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (act) {
          const int pos = nFG + __popc(bal & ltmask);
          const TmlSEnt dtl = LD_S(&s_tl[e]);
          FEnt<R> fe{};
          fe.off = x.off + LD_S(&s_coloff[x.cofs + (int)M]) - ((x.u ^ 1u) << 15);
          fe.J = (R)dtl.J;
          fe.fl = dtl.a * (uint32_t)nL * 2u;
          fe.uw = x.u << 15;
          ST_S(&FGl[pos], fe);
        }
        nFG += __popc(bal);
      }
      // pad the flip lists to a multiple of 4 with entries that are never active: row w of FLtab is
      // all zero, so (entry ^ 0) & 0x8000 == 0 for every lane
      if (lane < 4) {
        FEnt<R> z{}; z.off = cb; z.J = 0; z.fl = (uint32_t)p.w * (uint32_t)nL * 2u; z.uw = 0;
        { const uint32_t q = (nFS + lane); if (q < (uint32_t)((nFS + 3) & ~3)) ST_S(&FSl[q], z); }
        z.off = base + cb;
        { const uint32_t q = (nFG + lane); if (q < (uint32_t)((nFG + 3) & ~3)) ST_S(&FGl[q], z); }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) sumJ += __shfl_xor_sync(0xffffffffu, sumJ, o);
      const R dcoef = p.diag_coef - sumJ;
#if !defined(FTLM_NEG_TEST) || FTLM_NEG_TEST != 2     // (negative test of the host emulation: tests/emu/build_emu.py)
      __syncwarp();
#endif
      const int nFS4 = (nFS + 3) & ~3, nFG4 = (nFG + 3) & ~3;
      // ---- rows ------------------------------------------------------------------------------------
      const unsigned char* vsb = vsb0 + (size_t)cb * RB;                  // column base (bytes)
      for (int c = 0; c < nch; ++c) {
        const int lr = (chunk0 + c) * 32 + lane;
        const bool valid = lr < len;
        const int lrc = valid ? lr : 0;
        const int Lidx = k0 + lrc;
        const unsigned char* pl = vsb0 + (size_t)lrc * RB;               // lane pointer: row lrc of column 0
        const unsigned char* flp = s_fl + Lidx * 2;
        const V own = LD_S((const V*)(vsb + (size_t)lrc * RB));
        V qp;                                             // q_prev: issued now, consumed in the epilogue
        if (FUSED) qp = vec_ldcs(qprev + ((size_t)base + cb + lrc));
        V acc;
#pragma unroll
        for (int b = 0; b < B; ++b) acc.x[b] = dcoef * own.x[b];
        // U: same lr in another tile (TT) / another tile and column (TM): coalesced global reads (issued first)
        {
          const V* vl = v + lrc;
          int e = 0;
          for (; e + 4 <= nU; e += 4) {
            const UEnt<R> d0 = LD_S(&Ul[e]), d1 = LD_S(&Ul[e + 1]), d2 = LD_S(&Ul[e + 2]), d3 = LD_S(&Ul[e + 3]);
            const V a0 = vec_ldg((const V*)addr_u32(vl, d0.off, RB));
            const V a1 = vec_ldg((const V*)addr_u32(vl, d1.off, RB));
            const V a2 = vec_ldg((const V*)addr_u32(vl, d2.off, RB));
            const V a3 = vec_ldg((const V*)addr_u32(vl, d3.off, RB));
#pragma unroll
            for (int b = 0; b < B; ++b) acc.x[b] += d0.J * a0.x[b] + d1.J * a1.x[b] + d2.J * a2.x[b] + d3.J * a3.x[b];
          }
          for (; e < nU; ++e) {
            const UEnt<R> d = LD_S(&Ul[e]);
            const V a = vec_ldg((const V*)addr_u32(vl, d.off, RB));
#pragma unroll
            for (int b = 0; b < B; ++b) acc.x[b] += d.J * a.x[b];
          }
        }
        // FG: another tile, row flipped at L_i (per-lane test L_i != T_s); inactive lanes re-read nothing
        for (int e = 0; e < nFG4; e += 4) {
          uint32_t o0, o1, o2, o3, f0, f1, f2, f3, u0, u1, u2, u3;
          R j0, j1, j2, j3;
          load_fent(FGl + e, o0, j0, f0, u0); load_fent(FGl + e + 1, o1, j1, f1, u1);
          load_fent(FGl + e + 2, o2, j2, f2, u2); load_fent(FGl + e + 3, o3, j3, f3, u3);
          const uint32_t x0 = LD_S((const uint16_t*)(flp + f0)), x1 = LD_S((const uint16_t*)(flp + f1));
          const uint32_t x2 = LD_S((const uint16_t*)(flp + f2)), x3 = LD_S((const uint16_t*)(flp + f3));
          V a0 = own, a1 = own, a2 = own, a3 = own;
          if ((x0 ^ u0) & 0x8000u) a0 = vec_ldg((const V*)addr_u32(v, o0 + x0, RB));
          if ((x1 ^ u1) & 0x8000u) a1 = vec_ldg((const V*)addr_u32(v, o1 + x1, RB));
          if ((x2 ^ u2) & 0x8000u) a2 = vec_ldg((const V*)addr_u32(v, o2 + x2, RB));
          if ((x3 ^ u3) & 0x8000u) a3 = vec_ldg((const V*)addr_u32(v, o3 + x3, RB));
#pragma unroll
          for (int b = 0; b < B; ++b)
            acc.x[b] += j0 * (a0.x[b] - own.x[b]) + j1 * (a1.x[b] - own.x[b]) + j2 * (a2.x[b] - own.x[b]) + j3 * (a3.x[b] - own.x[b]);
        }
        // LL: swap form, 4 bonds per 8-byte table entry
        for (int g = 0; g < (p.n_ll4 >> 2); ++g) {
          const uint2 q = LD_S(&s_ll[g * nL + Lidx]);
          // a parallel (or padding) bond's table entry is the row itself: only the antiparallel lanes read
          // (fewer lanes per shared-memory wavefront, fewer bank conflicts: profiles/r02_emu_smem_profile.md)
          const uint32_t t0 = q.x & 0xffffu, t1 = q.x >> 16, t2 = q.y & 0xffffu, t3 = q.y >> 16;
          const V a0 = LD_S_IF(t0 != (uint32_t)lrc, (const V*)(vsb + t0 * RB), own);
          const V a1 = LD_S_IF(t1 != (uint32_t)lrc, (const V*)(vsb + t1 * RB), own);
          const V a2 = LD_S_IF(t2 != (uint32_t)lrc, (const V*)(vsb + t2 * RB), own);
          const V a3 = LD_S_IF(t3 != (uint32_t)lrc, (const V*)(vsb + t3 * RB), own);
          const R j0 = p.ll_J[4 * g + 0], j1 = p.ll_J[4 * g + 1], j2 = p.ll_J[4 * g + 2], j3 = p.ll_J[4 * g + 3];
#pragma unroll
          for (int b = 0; b < B; ++b) acc.x[b] += j0 * a0.x[b] + j1 * a1.x[b] + j2 * a2.x[b] + j3 * a3.x[b];
        }
        // S: other column of this tile, same lr
#pragma unroll 4
        for (int e = 0; e < nS; ++e) {
          const UEnt<R> d = LD_S(&Sl[e]);
          const V a = LD_S((const V*)(pl + d.off));
#pragma unroll
          for (int b = 0; b < B; ++b) acc.x[b] += d.J * a.x[b];
        }
        // FS: other column of this tile, row = L with bit i flipped (per-lane test L_i != M_j)
        for (int e = 0; e < nFS4; e += 4) {
          uint32_t o0, o1, o2, o3, f0, f1, f2, f3, u0, u1, u2, u3;
          R j0, j1, j2, j3;
          load_fent(FSl + e, o0, j0, f0, u0); load_fent(FSl + e + 1, o1, j1, f1, u1);
          load_fent(FSl + e + 2, o2, j2, f2, u2); load_fent(FSl + e + 3, o3, j3, f3, u3);
          const uint32_t x0 = LD_S((const uint16_t*)(flp + f0)), x1 = LD_S((const uint16_t*)(flp + f1));
          const uint32_t x2 = LD_S((const uint16_t*)(flp + f2)), x3 = LD_S((const uint16_t*)(flp + f3));
          const V a0 = LD_S_IF((x0 ^ u0) & 0x8000u, (const V*)(vsb0 + (size_t)(o0 + x0) * RB), own);
          const V a1 = LD_S_IF((x1 ^ u1) & 0x8000u, (const V*)(vsb0 + (size_t)(o1 + x1) * RB), own);
          const V a2 = LD_S_IF((x2 ^ u2) & 0x8000u, (const V*)(vsb0 + (size_t)(o2 + x2) * RB), own);
          const V a3 = LD_S_IF((x3 ^ u3) & 0x8000u, (const V*)(vsb0 + (size_t)(o3 + x3) * RB), own);
#pragma unroll
          for (int b = 0; b < B; ++b)
            acc.x[b] += j0 * (a0.x[b] - own.x[b]) + j1 * (a1.x[b] - own.x[b]) + j2 * (a2.x[b] - own.x[b]) + j3 * (a3.x[b] - own.x[b]);
        }
        // epilogue: Lanczos recurrence, reductions
        if (valid) {
          const size_t g = (size_t)base + cb + lrc;
          if (FUSED) {
#pragma unroll
            for (int b = 0; b < B; ++b) {
              acc.x[b] -= bprev.x[b] * qp.x[b];
              if (FUSED == 1) {
                s_qy[b] += (double)own.x[b] * (double)acc.x[b];
                s_yy[b] += (double)acc.x[b] * (double)acc.x[b];
                s_qq[b] += (double)own.x[b] * (double)own.x[b];
              }
            }
          }
          vec_stcs(y + g, acc);
        }
      }
    }
    if (FUSED == 1) {                                   // deterministic per-tile partial sums
#pragma unroll
      for (int b = 0; b < B; ++b) {
        const double a = warp_sum(s_qy[b]), bb = warp_sum(s_yy[b]), c = warp_sum(s_qq[b]);
        if (lane == 0) { ST_S(&S.red[warp * 3 * B + 3 * b], a); ST_S(&S.red[warp * 3 * B + 3 * b + 1], bb); ST_S(&S.red[warp * 3 * B + 3 * b + 2], c); }
      }
      __syncthreads();
      if (tid < 3 * B) {
        double s = 0.0;
        for (int wv = 0; wv < NW; ++wv) s += LD_S(&S.red[wv * 3 * B + tid]);
        ST_G(&p.partials[(size_t)tid * p.nT + T], s);
      }
    }
  }
  // ---- grid-wide finish: the last CTA resets the counters and (fused) advances the chains --------
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_last = (atomicAdd(&p.counter[1], 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (tid == 0) { p.counter[0] = 0; p.counter[1] = 0; }
  if (FUSED != 1) return;
  for (int q = 0; q < 3 * B; ++q) {                       // fixed assignment and order
    double a = 0.0;
    for (uint32_t k = tid; k < p.nT; k += NT) a += LD_G(&p.partials[(size_t)q * p.nT + k]);
    a = warp_sum(a);
    __syncthreads();
    if (lane == 0) ST_S(&S.red[warp], a);
    __syncthreads();
    if (tid == 0) {
      double s = 0.0;
      for (int wv = 0; wv < NW; ++wv) s += LD_S(&S.red[wv]);
      ST_S(&S.red[64 + q], s);
    }
  }
  __syncthreads();
  if (tid < B) {
    ChainState* st = p.st + tid;
    if (!st->done) {
      const double a = LD_S(&S.red[64 + 3 * tid]), b = LD_S(&S.red[64 + 3 * tid + 1]), c = LD_S(&S.red[64 + 3 * tid + 2]);
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
      if (j + 1 >= st->limit || beta <= st->tol * sc) { st->done = 1; st->inv_b = 0.0; }
    }
  }
}

// Neighbour indices through the TML tables (test hook; same tables, same base()/coloff/FLtab/LLtab
// arithmetic as hv_tml_kernel, read from global memory).  The row's own (T, M, L) comes from a full
// unrank and is cross-checked against the tables (a mismatch writes -2).
template <typename R, int MODE>
__global__ void __launch_bounds__(256)
neighbors_tml_kernel(const __grid_constant__ TmlParams<R> p, const BondDev* __restrict__ bonds, int nb,
                     const int* __restrict__ bclass, const int* __restrict__ bentry,
                     int64_t row0, int64_t nrows, int64_t* __restrict__ out) {
  const int K1 = p.K + 1;
  const int* koff = (const int*)(p.blob + p.off_koff);
  const uint16_t* coloff = (const uint16_t*)(p.blob + p.off_coloff);
  const uint2* ll = (const uint2*)(p.blob + p.off_ll);
  const uint16_t* fl = (const uint16_t*)(p.blob + p.off_fl);
  const TmlSEnt* mm = (const TmlSEnt*)(p.blob + p.off_mm);
  const TmlSEnt* ml = (const TmlSEnt*)(p.blob + p.off_ml);
  const TmlSEnt* tm = (const TmlSEnt*)(p.blob + p.off_tm);
  const TmlSEnt* tl = (const TmlSEnt*)(p.blob + p.off_tl);
  const int nL = 1 << p.w, nM = 1 << p.m;
  for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < nrows; r += (int64_t)gridDim.x * blockDim.x) {
    const uint64_t tr = (uint64_t)(row0 + r);
    uint64_t n = 0, rem = tr;
    int A = p.K;
    for (int q = p.N - 1; q >= 0 && A > 0; --q) {
      const uint64_t c = LD_G(&p.binom[q * K1 + A]);
      if (rem >= c) { n |= 1ull << q; rem -= c; --A; }
    }
    const uint32_t T = (uint32_t)(n >> p.mw), M = (uint32_t)(n >> p.w) & (uint32_t)(nM - 1), L = (uint32_t)n & (uint32_t)(nL - 1);
    const int kT = p.K - __popc(T), kL = kT - __popc(M);
    const uint64_t base = tml_base<MODE>(T, p.mw, p.K, p.binom, p.clt);
    const int cb = (kT >= 0 && kT <= p.mw) ? (int)LD_G(&coloff[kT * nM + M]) : 0;
    const int lr = (int)(tr - base) - cb;
    bool ok = kL >= 0 && kL <= p.w && lr >= 0 && lr < LD_G(&koff[kL + 1]) - LD_G(&koff[kL]);
    const int Lidx = ok ? LD_G(&koff[kL]) + lr : 0;
    for (int i = 0; ok && i < p.w; ++i) ok = ((LD_G(&fl[i * nL + Lidx]) >> 15) == ((L >> i) & 1u));   // FLtab knows L
    for (int b = 0; b < nb; ++b) {
      const uint64_t mk = LD_G(&bonds[b].mask), x = n & mk;
      int64_t idx = -1;
      const int e = LD_G(&bentry[b]), bcls = LD_G(&bclass[b]);
      if (x != 0 && x != mk) {
        switch (bcls) {
          case 0: {                                      // LL
            const uint2 q = LD_G(&ll[(e >> 2) * nL + Lidx]);
            const uint32_t h = (e & 2) ? q.y : q.x;
            idx = (int64_t)base + cb + (int)((e & 1) ? (h >> 16) : (h & 0xffffu));
            break;
          }
          case 1: idx = (int64_t)base + LD_G(&coloff[kT * nM + (M ^ LD_G(&mm[e].a))]) + lr; break;                 // MM
          case 2: idx = (int64_t)base + LD_G(&coloff[kT * nM + (M ^ (1u << LD_G(&ml[e].b)))]) +        // ML
                        (int)(LD_G(&fl[LD_G(&ml[e].a) * nL + Lidx]) & 0x7fffu); break;
          case 3: idx = (int64_t)tml_base<MODE>(T ^ p.tt_mask[e & (TML_MAX_TT - 1)], p.mw, p.K, p.binom, p.clt) + cb + lr; break;  // TT
          case 6: {                                      // PASS-B window e: run start of the swapped window word + offset in the run
            const int lo = p.pb_lo[e & 7];
            const uint64_t hi = n >> lo, low = n & ((1ull << lo) - 1ull);
            const int kP = p.K - __popcll((unsigned long long)hi);
            const uint64_t x = passb_low_rank(low, p.K, p.binom);
            const uint64_t own = passb_run_start<MODE>(hi, lo, kP, p.K, p.binom, p.clt);
            idx = (int64_t)(passb_run_start<MODE>(hi ^ (mk >> lo), lo, kP, p.K, p.binom, p.clt) + x);
            if (own + x != tr) idx = -4;                 // the run arithmetic must reproduce the row's own index
            break;
          }
          default: {                                     // TM / TL
            const TmlSEnt d = bcls == 4 ? LD_G(&tm[e]) : LD_G(&tl[e]);
            const uint32_t bit = 1u << p.ts_site[d.b & (TML_MAX_TS - 1)];
            const int kTp = (T & bit) ? kT + 1 : kT - 1;
            const uint64_t tb = tml_base<MODE>(T ^ bit, p.mw, p.K, p.binom, p.clt);
            if (kTp < 0 || kTp > p.mw) idx = -5;         // cannot happen for an antiparallel bond
            else if (bcls == 4) idx = (int64_t)tb + LD_G(&coloff[kTp * nM + (M ^ (1u << d.a))]) + lr;
            else idx = (int64_t)tb + LD_G(&coloff[kTp * nM + M]) + (int)(LD_G(&fl[d.a * nL + Lidx]) & 0x7fffu);
          }
        }
        if (!ok) idx = -2;
      } else if (bcls == 0 && ok) {                 // parallel LL bond: the table must say "self"
        const uint2 q = LD_G(&ll[(e >> 2) * nL + Lidx]);
        const uint32_t h = (e & 2) ? q.y : q.x;
        if ((int)((e & 1) ? (h >> 16) : (h & 0xffffu)) != lr) idx = -3;
      }
      ST_G(&out[r * nb + b], idx);
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
void fill_params(const ftlm_ctx* c, const TmlPlan* t, TmlParams<R>& p, int batch) {
  memset(&p, 0, sizeof(p));
  p.N = c->N; p.K = c->N_up; p.w = t->w; p.m = t->m; p.t = t->t; p.mw = t->w + t->m; p.mode = c->mode;
  p.nT = t->nT; p.t_begin = 0; p.t_end = t->nT;
  if (c->debug_item_count > 0) {
    p.t_begin = (uint32_t)std::min<int64_t>(c->debug_item_first, t->nT);
    p.t_end = (uint32_t)std::min<int64_t>(c->debug_item_first + c->debug_item_count, t->nT);
  }
  p.n_ll4 = t->n_ll4; p.n_mm = t->n_mm; p.n_ml = t->n_ml; p.n_tt = t->n_tt; p.n_ts = t->n_ts;
  p.n_tm = t->n_tm; p.n_tl = t->n_tl;
  p.max_tile = t->max_tile;
  p.scratch_bytes = tml_scratch_bytes((int)sizeof(R), t->n_tt, t->n_tm, t->n_mm, t->n_ml, t->n_tl);
  p.dim = c->dim; p.binom = c->d_binom64; p.clt = c->d_clt; p.blob = t->d_blob;
  p.blob_bytes = t->blob_bytes; p.off_koff = t->off_koff; p.off_tlen = t->off_tlen; p.off_coloff = t->off_coloff;
  p.off_ll = t->off_ll; p.off_fl = t->off_fl; p.off_mm = t->off_mm; p.off_ml = t->off_ml; p.off_tm = t->off_tm;
  p.off_tl = t->off_tl; p.items = t->d_items; p.item_off = t->d_item_off;
  p.partials = t->d_partials; p.counter = t->d_counter; p.st = c->d_state; p.diag_coef = (R)t->diag_coef;
  for (int k = 0; k < t->n_ll4; ++k) p.ll_J[k] = (R)t->ll_J[(size_t)k];
  for (int k = 0; k < t->n_tt; ++k) { p.tt_mask[k] = t->tt_mask[(size_t)k]; p.tt_J[k] = t->tt_J[(size_t)k]; }
  for (int k = 0; k < t->n_ts; ++k) p.ts_site[k] = t->ts_site[(size_t)k];
  for (int k = 0; k < 8 && k < ftlm_passb_windows(c); ++k) { int lo, sz; ftlm_passb_window_geometry(c, k, &lo, &sz); p.pb_lo[k] = lo; }
  (void)batch;
}

struct TmlLaunchCfg { int threads, ctas; size_t smem; };

// threads / CTAs per SM / dynamic shared memory for a batch of B vectors; smem == 0 if it does not fit
TmlLaunchCfg tml_config(const ftlm_ctx* c, const TmlPlan* t, int batch) {
  const int esz = (int)ftlm_elem_size(c);
  const int sb = tml_scratch_bytes(esz, t->n_tt, t->n_tm, t->n_mm, t->n_ml, t->n_tl);
  const size_t cap = 227 * 1024 - 1024;
  TmlSmem S;
  TmlLaunchCfg best{0, 0, 0};
  const size_t s512 = tml_layout(S, nullptr, c->N, c->N_up, t->blob_bytes, t->max_tile, esz * batch, batch, 16, sb);
  if (batch < 4) {
    if (2 * (s512 + 1024) <= 228 * 1024) return TmlLaunchCfg{512, 2, s512};
    const size_t s1024 = tml_layout(S, nullptr, c->N, c->N_up, t->blob_bytes, t->max_tile, esz * batch, batch, 32, sb);
    if (s1024 <= cap) return TmlLaunchCfg{1024, 1, s1024};
  }
  if (s512 <= cap) return TmlLaunchCfg{512, (2 * (s512 + 1024) <= 228 * 1024) ? 2 : 1, s512};
  return best;
}

template <typename R, int B, int MODE>
int launch_tml(ftlm_ctx* c, const void* v, const void* qp, void* y, int fused, cudaStream_t s) {
  TmlPlan* t = c->tml;
  // launch shape of the batch the plan was built for: a narrower run on the same plan (remainder group, plan_batch)
  // keeps the thread count and hence the order of every sum
  const TmlLaunchCfg cfg = tml_config(c, t, std::max(B, ftlm_plan_batch(c)));
  if (cfg.smem == 0) { ftlm_set_error("TML: batch %d does not fit shared memory with this split", B); return FTLM_EUNSUPPORTED; }
  if (fused == 1 && B > t->partials_batch) { ftlm_set_error("TML: internal: partials sized for batch %d", t->partials_batch); return FTLM_EINVAL; }
  TmlParams<R> p;
  fill_params<R>(c, t, p, B);
  int grid = c->sm_count * cfg.ctas;
  if ((uint32_t)grid > p.t_end - p.t_begin) grid = (int)std::max(1u, p.t_end - p.t_begin);
  if (fused == 1) {
    auto k = hv_tml_kernel<R, B, MODE, 1>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem));
    FTLM_LAUNCH(k, grid, cfg.threads, cfg.smem, s, p, (const R*)v, (const R*)qp, (R*)y);
  } else if (fused == 2) {
    auto k = hv_tml_kernel<R, B, MODE, 2>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem));
    FTLM_LAUNCH(k, grid, cfg.threads, cfg.smem, s, p, (const R*)v, (const R*)qp, (R*)y);
  } else {
    auto k = hv_tml_kernel<R, B, MODE, 0>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem));
    FTLM_LAUNCH(k, grid, cfg.threads, cfg.smem, s, p, (const R*)v, (const R*)qp, (R*)y);
  }
  CK(cudaGetLastError());
  return FTLM_OK;
}

template <typename R, int MODE>
int launch_tml_b(ftlm_ctx* c, const void* v, const void* qp, void* y, int fused, int batch, cudaStream_t s) {
  switch (batch) {
    case 1: return launch_tml<R, 1, MODE>(c, v, qp, y, fused, s);
    case 2: return launch_tml<R, 2, MODE>(c, v, qp, y, fused, s);
    case 4: return launch_tml<R, 4, MODE>(c, v, qp, y, fused, s);
    default: ftlm_set_error("TML: batch must be 1, 2 or 4 (got %d)", batch); return FTLM_EINVAL;
  }
}

}  // namespace

void ftlm_tml_plan_destroy(ftlm_ctx* c) {
  ftlm_passb_plan_destroy(c);
  ftlm_tmlr_plan_destroy(c);
  TmlPlan* t = c->tml;
  if (!t) return;
  ftlm_dfree(t->d_blob); ftlm_dfree(t->d_items); ftlm_dfree(t->d_item_off); ftlm_dfree(t->d_partials);
  ftlm_dfree(t->d_counter); ftlm_dfree(t->d_bond_class); ftlm_dfree(t->d_bond_entry);
  delete t;
  c->tml = nullptr;
}

// Build the plan.  FTLM_OK with c->tml == nullptr when no split is possible for this sector (the
// dispatcher then uses the TILE / ROW kernels).  c->tml_low_bits / c->tml_mid_bits (0 = auto) choose w, m.
static int tml_plan_try(ftlm_ctx* c, int w, int m, bool forced);

int ftlm_tml_plan_create(ftlm_ctx* c) {
  c->tml = nullptr;
  if (c->mode == FTLM_INDEX_LIN) return FTLM_OK;       // Lin tables serve the thread-per-row kernel only
  const int N = c->N;
  const bool forced = c->tml_low_bits != 0 || c->tml_mid_bits != 0;
  if (forced) return tml_plan_try(c, c->tml_low_bits ? c->tml_low_bits : 9, c->tml_mid_bits ? c->tml_mid_bits : 7, true);
  // auto: the largest tile that fits shared memory (fewer bonds leave the tile), w = 9 low bits
  for (int mw = N - 6 < 17 ? N - 6 : 17; mw >= 6; --mw) {
    const int w = mw - 2 < 9 ? mw - 2 : 9;
    int rc = tml_plan_try(c, w, mw - w, false);
    if (rc != FTLM_OK) return rc;
    if (c->tml) break;
  }
  return FTLM_OK;
}

static int tml_plan_try(ftlm_ctx* c, int w, int m, bool forced) {
  c->tml = nullptr;
  const int N = c->N, esz = (int)ftlm_elem_size(c);
  const int t = N - w - m;
  auto unusable = [&](const char* why) {
    if (forced) { ftlm_set_error("TML: low_bits=%d mid_bits=%d unusable for N=%d: %s", w, m, N, why); return (int)FTLM_EUNSUPPORTED; }
    return (int)FTLM_OK;
  };
  // t <= 22: the per-tile partial sums (96 bytes per top part and chain) and the tile counter stay small; sparse
  // sectors of very long labels (N = 46..48 with few up spins) fall back to the ROW kernel instead of asking for 10^11 bytes
  if (w < 5 || w > 12 || m < 1 || m > 9 || w + m > 18 || t < 1 || t > 22) return unusable("need 5<=w<=12, 1<=m<=9, w+m<=18, 1<=t<=22");
  if (c->dim < 64) return unusable("sector too small");
  if ((uint64_t)c->dim >= (1ull << 32)) return unusable("dim >= 2^32 (row offsets are 32-bit)");
  const int mw = w + m;
  TmlPlan* P = new TmlPlan();
  P->w = w; P->m = m; P->t = t; P->nT = 1u << t;
  std::vector<int> bclass((size_t)c->nb, 0), bentry((size_t)c->nb, 0);
  struct LLb { uint32_t mask; double Jh; };
  std::vector<LLb> ll;
  std::vector<int> ts_index((size_t)t, -1);
  auto ts_of = [&](int site) {
    const int s = site - mw;
    if (ts_index[(size_t)s] < 0) { ts_index[(size_t)s] = (int)P->ts_site.size(); P->ts_site.push_back((uint8_t)s); }
    return (uint32_t)ts_index[(size_t)s];
  };
  double sumJ_ll = 0.0;
  // bonds that leave the tile (a site at or above mw): PASS-B windows take what they can cover
  // (class 6, entry = window); the rest is read from global memory here (TT / TM / TL)
  std::vector<int> cand, window_of;
  for (int b = 0; b < c->nb; ++b) if (c->bonds[(size_t)b].j >= mw) cand.push_back(b);
  {
    ftlm_passb_plan_destroy(c);
    int rc = ftlm_passb_plan_create(c, mw, cand, window_of);
    if (rc != FTLM_OK) { delete P; return rc; }
  }
  std::vector<int> win_of_bond((size_t)c->nb, -1);
  for (size_t k = 0; k < cand.size(); ++k) win_of_bond[(size_t)cand[k]] = window_of[k];
  for (int b = 0; b < c->nb; ++b) {
    const BondDev& d = c->bonds[(size_t)b];
    const int i = d.i, j = d.j;                                          // i < j
    if (win_of_bond[(size_t)b] >= 0) { bclass[(size_t)b] = 6; bentry[(size_t)b] = win_of_bond[(size_t)b]; }
    else if (j < w) { bclass[(size_t)b] = 0; bentry[(size_t)b] = (int)ll.size(); ll.push_back({(uint32_t)d.mask, d.Jh}); sumJ_ll += d.Jh; }
    else if (i >= w && j < mw) { bclass[(size_t)b] = 1; bentry[(size_t)b] = (int)P->mm.size(); P->mm.push_back({(uint32_t)(d.mask >> w), 0u, d.Jh}); }
    else if (i < w && j < mw) { bclass[(size_t)b] = 2; bentry[(size_t)b] = (int)P->ml.size(); P->ml.push_back({(uint32_t)i, (uint32_t)(j - w), d.Jh}); }
    else if (i >= mw) { bclass[(size_t)b] = 3; bentry[(size_t)b] = (int)P->tt_mask.size(); P->tt_mask.push_back((uint32_t)(d.mask >> mw)); P->tt_J.push_back(d.Jh); }
    else if (i >= w) { bclass[(size_t)b] = 4; bentry[(size_t)b] = (int)P->tm.size(); P->tm.push_back({(uint32_t)(i - w), ts_of(j), d.Jh}); }
    else { bclass[(size_t)b] = 5; bentry[(size_t)b] = (int)P->tl.size(); P->tl.push_back({(uint32_t)i, ts_of(j), d.Jh}); }
  }
  P->n_ll = (int)ll.size(); P->n_ll4 = (P->n_ll + 3) & ~3;
  P->n_mm = (int)P->mm.size(); P->n_ml = (int)P->ml.size(); P->n_tt = (int)P->tt_mask.size();
  P->n_ts = (int)P->ts_site.size(); P->n_tm = (int)P->tm.size(); P->n_tl = (int)P->tl.size();
  if (P->n_ll4 > TML_MAX_LL || P->n_mm > TML_MAX_LIST || P->n_ml > TML_MAX_LIST || P->n_tt > TML_MAX_TT ||
      P->n_ts > TML_MAX_TS || P->n_tm > TML_MAX_LIST || P->n_tl > TML_MAX_LIST) { ftlm_passb_plan_destroy(c); delete P; return unusable("too many bonds in one class"); }
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
  if (P->max_tile > 65535 || binom_t(w, w / 2) > 32767) { ftlm_passb_plan_destroy(c); delete P; return unusable("tile too large for 16-bit offsets"); }
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
      const int nchunks = (len + 31) / 32;
      for (int ch = 0; ch < nchunks; ch += TML_MAX_CHUNKS) {
        const int nc = std::min(TML_MAX_CHUNKS, nchunks - ch);
        items.push_back((uint32_t)M | ((uint32_t)ch << 16) | ((uint32_t)nc << 24));
      }
      off += len;
    }
    // longest columns first: the strided assignment item -> warp then balances the warps
    std::stable_sort(items.begin() + item_off[(size_t)kT], items.end(),
                     [](uint32_t a, uint32_t b) { return (a >> 24) > (b >> 24); });
    item_off[(size_t)kT + 1] = (int)items.size();
  }
  std::vector<uint16_t> lltab((size_t)(P->n_ll4 / 4) * nL * 4, 0), fltab((size_t)(w + 1) * nL, 0);   // row w stays zero (padding entries)
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
        lltab[((size_t)(b >> 2) * nL + Lidx) * 4 + (b & 3)] = (uint16_t)nb;
      }
      for (int i = 0; i < w; ++i)
        fltab[(size_t)i * nL + Lidx] = (uint16_t)((uint32_t)lr[(size_t)(L ^ (1u << i))] | (((L >> i) & 1u) << 15));
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
  P->off_coloff = put(coloff.data(), coloff.size() * 2);
  P->off_ll = put(lltab.data(), lltab.size() * 2);
  P->off_fl = put(fltab.data(), fltab.size() * 2);
  P->off_mm = put(P->mm.data(), P->mm.size() * sizeof(TmlSEnt));
  P->off_ml = put(P->ml.data(), P->ml.size() * sizeof(TmlSEnt));
  P->off_tm = put(P->tm.data(), P->tm.size() * sizeof(TmlSEnt));
  P->off_tl = put(P->tl.data(), P->tl.size() * sizeof(TmlSEnt));
  P->blob_bytes = (int)blob.size();
  P->h_bond_class = bclass; P->h_bond_entry = bentry;
  c->tml = P;
  if (tml_config(c, P, ftlm_plan_batch(c)).smem == 0) { c->tml = nullptr; ftlm_passb_plan_destroy(c); delete P; return unusable("tables + tile exceed shared memory"); }
  // ---- upload ----------------------------------------------------------------------------------
  P->partials_batch = 4;
  auto up = [&](void** d, const void* h, size_t bytes) -> bool {
    if (ftlm_dmalloc(d, bytes ? bytes : 16) != cudaSuccess) return false;
    if (bytes && h && cudaMemcpy(*d, h, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return false;
    return true;
  };
  const size_t pbytes = (size_t)P->nT * 24 * (size_t)P->partials_batch;
  bool ok = up((void**)&P->d_blob, blob.data(), blob.size()) && up((void**)&P->d_items, items.data(), items.size() * 4) &&
            up((void**)&P->d_item_off, item_off.data(), item_off.size() * 4) &&
            up((void**)&P->d_bond_class, bclass.data(), bclass.size() * 4) &&
            up((void**)&P->d_bond_entry, bentry.data(), bentry.size() * 4) &&
            up((void**)&P->d_partials, nullptr, pbytes) && up((void**)&P->d_counter, nullptr, 16);
  if (ok) ok = cudaMemset(P->d_partials, 0, pbytes) == cudaSuccess && cudaMemset(P->d_counter, 0, 16) == cudaSuccess;
  if (!ok) { cudaGetLastError(); ftlm_tml_plan_destroy(c); ftlm_set_error("TML: table upload failed"); return FTLM_ENOMEM; }
  {                                                       // the register-table variant of the in-tile pass, when it applies
    std::vector<int> in_window((size_t)c->nb, 0);
    for (int b = 0; b < c->nb; ++b) in_window[(size_t)b] = win_of_bond[(size_t)b] >= 0 ? 1 : 0;
    int rc = ftlm_tmlr_plan_create(c, w, m, in_window);
    if (rc != FTLM_OK) { ftlm_tml_plan_destroy(c); return rc; }
  }
  return FTLM_OK;
}

int64_t ftlm_tml_info(const ftlm_ctx* c, const char* key) {
  const TmlPlan* t = c->tml;
  if (!t) return -1;
  if (!strcmp(key, "tml_w")) return t->w;
  if (!strcmp(key, "tml_tiles")) return (int64_t)t->nT;
  if (!strncmp(key, "tml_bclass:", 11)) {                 // class | entry << 8 of bond b (class 6 = PASS-B window `entry`)
    const int b = atoi(key + 11);
    if (b < 0 || b >= (int)t->h_bond_class.size()) return -1;
    return (int64_t)t->h_bond_class[(size_t)b] | ((int64_t)t->h_bond_entry[(size_t)b] << 8);
  }
  if (!strcmp(key, "tml_m")) return t->m;
  if (!strcmp(key, "tml_smem")) return (int64_t)tml_config(c, t, c->batch).smem;
  if (!strcmp(key, "tml_ctas_per_sm")) return tml_config(c, t, c->batch).ctas;
  if (!strcmp(key, "tml_threads")) return tml_config(c, t, c->batch).threads;
  if (!strcmp(key, "tml_max_batch")) { int b = 4; while (b > 1 && tml_config(c, t, b).smem == 0) b >>= 1; return b; }
  if (!strcmp(key, "tml_n_ll")) return t->n_ll;
  if (!strcmp(key, "tml_n_mm")) return t->n_mm;
  if (!strcmp(key, "tml_n_ml")) return t->n_ml;
  if (!strcmp(key, "tml_n_tt")) return t->n_tt;
  if (!strcmp(key, "tml_n_tm")) return t->n_tm;
  if (!strcmp(key, "tml_n_tl")) return t->n_tl;
  return -1;
}

int ftlm_launch_hv_tml(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, int batch, cudaStream_t s) {
  if (!c->tml) { ftlm_set_error("TML kernel unavailable"); return FTLM_EUNSUPPORTED; }
  if (c->prec == FTLM_FP32) {
    if (c->mode == FTLM_INDEX_CLT) return launch_tml_b<float, FTLM_INDEX_CLT>(c, v, qprev, y, fused, batch, s);
    return launch_tml_b<float, FTLM_INDEX_CR>(c, v, qprev, y, fused, batch, s);
  }
  if (c->mode == FTLM_INDEX_CLT) return launch_tml_b<double, FTLM_INDEX_CLT>(c, v, qprev, y, fused, batch, s);
  return launch_tml_b<double, FTLM_INDEX_CR>(c, v, qprev, y, fused, batch, s);
}

int ftlm_launch_neighbors_tml(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s) {
  TmlPlan* t = c->tml;
  if (!t) { ftlm_set_error("TML kernel unavailable"); return FTLM_EUNSUPPORTED; }
  int64_t blocks = (nrows + 255) / 256;
  if (blocks > c->sm_count * 8) blocks = c->sm_count * 8;
#define LAUNCHN(R, MODE)                                                                                   \
  do {                                                                                                     \
    TmlParams<R> p;                                                                                        \
    fill_params<R>(c, t, p, 1);                                                                            \
    { auto k__ = neighbors_tml_kernel<R, MODE>; FTLM_LAUNCH(k__, (int)blocks, 256, 0, s, p, c->d_bonds, c->nb, t->d_bond_class,        \
                                                               t->d_bond_entry, row0, nrows, d_idx); }       \
  } while (0)
  if (c->prec == FTLM_FP32) { if (c->mode == FTLM_INDEX_CLT) LAUNCHN(float, FTLM_INDEX_CLT); else LAUNCHN(float, FTLM_INDEX_CR); }
  else { if (c->mode == FTLM_INDEX_CLT) LAUNCHN(double, FTLM_INDEX_CLT); else LAUNCHN(double, FTLM_INDEX_CR); }
#undef LAUNCHN
  CK(cudaGetLastError());
  return FTLM_OK;
}
