// TMLR kernel - the in-tile pass of the gather H.v with lane tables held in registers
// (DESIGN.md section 6.5).  Same label split as the TML kernel, n = (T | M | L), same tile in shared
// memory, same index arithmetic (index = base(T) + coloff[kT][M] + lr(L); base(T) by CR - Alg. 1
// restricted to the top bits - or by CLT - Alg. 2 with j = 0), but the loops are turned inside out:
// a warp keeps one chunk of 32 low parts L (fixed popcount kL, lane <-> lr) and walks over the
// columns M of matching popcount.  Everything that depends on L alone - the target row of every LL
// bond, the flipped row and the spin L_i of every ML bond - is read once per unit into registers;
// everything that depends on M alone - the diagonal coefficient, the antiparallel MM bonds and their
// target columns, the target column and the spin M_j of every ML bond - is a descriptor built once
// per tile in shared memory.  Per row and bond the inner loops are then
//   LL:  one shared-memory read + one FMA             (swap form: parallel bonds read the row itself)
//   MM:  one descriptor read (warp-uniform), one shared-memory read, one FMA, antiparallel bonds only
//   ML:  one descriptor read (warp-uniform), a lane test L_i != M_j, one predicated read, one FMA.
// (Eq. 12 with the s = 1/2 coefficients of Eqs. 13-14 in swap form, y_t = d0 v_t + sum_b (J_b/2)(v[P_b n_t] - v_t)).
// The bonds that leave the tile belong to the PASS-B windows; a few left-over ones that are uniform per
// column (both sites in T, or one in T and one in M) are read from global memory at the same lr (coalesced);
// the plan is refused if a left-over bond has a site in L (that needs the TML kernel's per-lane gather).
#include <algorithm>
#include <cstring>
#include <vector>

#define FTLM_TU 4
#include "ftlm_passb.cuh"

#define TMLR_MAX_LL 16
#define TMLR_MAX_MM 16
#define TMLR_MAX_ML 16
#define TMLR_MAX_G 8              // bonds that leave the tile but are uniform per column (TT, TM): coalesced global reads
#define TMLR_THREADS 512

template <typename R>
struct TmlrParams {
  int N, K, w, m, mw;
  uint32_t nT, t_begin, t_end;
  int n_ll, n_mm, n_ml, max_tile;     // n_ll, n_ml: padded to multiples of 4 (the kernel's NLL, NML)
  int mode, fused;
  int lazy;                           // 1: the tile is formed from (vio = y_j, qprev = q_j) as (y_j - alpha_j q_j) / beta_j and written back to vio
  R* vio;
  int64_t dim;
  const uint64_t* binom;              // [(N+1)*(K+1)] global
  const uint2* clt;
  const unsigned char* blob;          // static tables, staged once per CTA
  int blob_bytes, off_koff, off_tlen, off_coloff, off_mlist, off_moff, off_ll, off_fl;
  const uint32_t* units;              // kL | chunk << 4 | col_begin << 8 | ncols << 20, grouped by kT
  const int* unit_off;                // [mw + 2]
  double* partials;                   // [3][nT]
  unsigned int* counter;              // [0] tile counter, [1] ticket
  ChainState* st;
  R coef0;                            // diag0 - sum of J_b/2 over the LL and ML bonds
  R ll_J[TMLR_MAX_LL], ml_J[TMLR_MAX_ML], mm_J[TMLR_MAX_MM];
  uint32_t mm_mask[TMLR_MAX_MM];
  int ml_j[TMLR_MAX_ML];              // M bit of ML bond e
  int n_g;                            // left-over bonds with a site in T and none in L
  uint32_t g_tmask[TMLR_MAX_G];       // T bits the bond flips (two for TT, one for TM)
  int g_mbit[TMLR_MAX_G];             // M bit of a TM bond, -1 for TT
  R g_J[TMLR_MAX_G];
};

struct TmlrPlan {
  int w = 0, m = 0, n_ll = 0, n_mm = 0, n_ml = 0, max_tile = 0;
  uint32_t nT = 0;
  unsigned char* d_blob = nullptr;
  int blob_bytes = 0, off_koff = 0, off_tlen = 0, off_coloff = 0, off_mlist = 0, off_moff = 0, off_ll = 0, off_fl = 0;
  uint32_t* d_units = nullptr;
  int* d_unit_off = nullptr;
  double* d_partials = nullptr;
  unsigned int* d_counter = nullptr;
  double coef0 = 0.0;
  std::vector<double> ll_J, ml_J, mm_J;
  std::vector<uint32_t> mm_mask;
  std::vector<int> ml_j;
  std::vector<uint32_t> g_tmask;
  std::vector<int> g_mbit;
  std::vector<double> g_J;
  int n_g = 0;
  size_t smem = 0;
  bool unij = false;                  // uniform J_b within the LL bonds and within the ML bonds
};

namespace {

// antiparallel MM bond of a column: row offset of the target column and J/2, read with one (broadcast) load
template <typename R> struct MmEnt;
template <> struct __align__(8) MmEnt<float> { uint32_t off; float J; };
template <> struct __align__(16) MmEnt<double> { uint32_t off, pad; double J; };

// per-column descriptor arrays in shared memory (rebuilt for every tile: they depend on kT)
template <typename R>
struct TmlrSmem {
  uint64_t* binom;
  unsigned char* blob;
  R* vs;                // tile
  R* dcoef;             // [nM] diagonal coefficient of column M
  MmEnt<R>* dmm;        // [nM][n_mm] antiparallel MM bonds (compacted): row offset of the target column, J/2
  uint32_t* dml;        // [nM][n_ml] byte offset of the target column | M_j (bit 0)
  int* dnmm;            // [nM]
  uint32_t* dg;         // [nM][n_g] global row (target tile base + target column offset) of the active left-over bonds
  R* dgJ;               // [nM][n_g]
  int* dng;             // [nM]
  double* red;          // [warps][3] + 3
  int* misc;            // [0] tile
};

template <typename R>
__host__ __device__ inline size_t tmlr_layout(TmlrSmem<R>& s, unsigned char* p0, int N, int K, int blob_bytes, int max_tile,
                                              int nM, int n_mm, int n_ml, int n_g, int warps) {
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 15) & ~(size_t)15; return p0 + at; };
  s.binom = (uint64_t*)take((size_t)(N + 1) * (K + 1) * 8);
  s.blob = take((size_t)blob_bytes);
  s.vs = (R*)take((size_t)max_tile * sizeof(R) + 16);    // + 16: the tile keeps the global address's residue mod 16 bytes
  s.dcoef = (R*)take((size_t)nM * sizeof(R));
  s.dmm = (MmEnt<R>*)take((size_t)nM * (n_mm ? n_mm : 1) * sizeof(MmEnt<R>));
  s.dml = (uint32_t*)take((size_t)nM * (n_ml ? n_ml : 1) * 4);
  s.dnmm = (int*)take((size_t)nM * 4);
  s.dg = (uint32_t*)take((size_t)nM * (n_g ? n_g : 1) * 4);
  s.dgJ = (R*)take((size_t)nM * (n_g ? n_g : 1) * sizeof(R));
  s.dng = (int*)take((size_t)nM * 4);
  s.red = (double*)take((size_t)(warps + 1) * 3 * 8);
  s.misc = (int*)take(16);
  return o;
}

}  // namespace

namespace {

// FUSED: 0 = y = H_A v;  1 = fused Lanczos pass (subtract beta q_prev, FP64 sums, finish);
//        2 = first pass of a multi-pass step: subtract beta q_prev only (the last PASS-B window finishes).
// NLL / NML: LL and ML bond slots (the plan pads the bond lists to multiples of 4 with J = 0 entries that
// read the row itself, so the inner loops carry no predicates).  mode / fused are warp-uniform run-time values.
// UNIJ: every LL bond has the same J_b and every ML bond has the same J_b (uniform-J lattices): the loops
// add the gathered values and multiply once (padding entries then add J * v_t, which coef0 takes back).
template <typename R, int NLL, int NML, bool UNIJ>
__global__ void __launch_bounds__(TMLR_THREADS, 1)
hv_tmlr_kernel(const __grid_constant__ TmlrParams<R> p, const R* __restrict__ v, const R* __restrict__ qprev,
               R* __restrict__ y) {
  FTLM_DYN_SMEM(smem);
  __shared__ bool s_last;
  const int FUSED = p.fused;
  if (FUSED && p.st->done) return;
  const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
  const int nL = 1 << p.w, nM = 1 << p.m;
  TmlrSmem<R> S;
  tmlr_layout<R>(S, smem, p.N, p.K, p.blob_bytes, p.max_tile, nM, p.n_mm, p.n_ml, p.n_g, NW);
  for (int k = tid; k < (p.N + 1) * (p.K + 1); k += NT) ST_S(&S.binom[k], LD_G(&p.binom[k]));
  {
    const uint4* src = (const uint4*)p.blob;
    uint4* dst = (uint4*)S.blob;
    for (int k = tid; k < (p.blob_bytes >> 4); k += NT) ST_S(&dst[k], LDG(&src[k]));
  }
  const int* s_koff = (const int*)(S.blob + p.off_koff);
  const int* s_tlen = (const int*)(S.blob + p.off_tlen);
  const uint16_t* s_coloff = (const uint16_t*)(S.blob + p.off_coloff);       // [kT][M]
  const uint16_t* s_mlist = (const uint16_t*)(S.blob + p.off_mlist);         // M sorted by popcount
  const int* s_moff = (const int*)(S.blob + p.off_moff);                     // [m+2]
  const uint16_t* s_ll = (const uint16_t*)(S.blob + p.off_ll);               // [bond][Lidx]: target row in the column
  const uint16_t* s_fl = (const uint16_t*)(S.blob + p.off_fl);               // [bond][Lidx]: flipped row | L_i << 15
  const R bprev = FUSED ? (R)p.st->beta_prev : (R)0;
  const int n_mm = p.n_mm;
  constexpr int n_ml = NML;
  constexpr int RPV = 16 / (int)sizeof(R);              // rows per 16 bytes
  __shared__ __align__(8) uint64_t s_mbar;              // completion barrier of the tile's bulk copy
  uint32_t mbar_parity = 0;
  if (tid == 0) mbar_init(&s_mbar, 1);

  if (tid == 0) S.misc[0] = (int)atomicAdd(&p.counter[0], 1u);
  for (;;) {
    __syncthreads();                                   // previous tile done (tile and descriptors reusable), next tile id visible
    const uint32_t T = (uint32_t)S.misc[0] + p.t_begin;
    __syncthreads();                                   // everyone has read it
    if (T >= p.t_end) break;
    if (tid == 0) S.misc[0] = (int)atomicAdd(&p.counter[0], 1u);   // the following tile's id travels while this tile is processed
    const int kT = p.K - __popc(T);
    if (kT < 0 || kT > p.mw) continue;                  // no rows with this top part
    const uint64_t base = p.mode == FTLM_INDEX_CLT ? passb_run_start<FTLM_INDEX_CLT>((uint64_t)T, p.mw, kT, p.K, S.binom, p.clt)
                                                   : passb_run_start<FTLM_INDEX_CR>((uint64_t)T, p.mw, kT, p.K, S.binom, p.clt);
    const int tlen = LD_S(&s_tlen[kT]);
    // the tile sits in shared memory at the same residue mod 16 bytes as in global memory, so that its 16-byte
    // aligned interior is one bulk copy (cp.async.bulk, SASS UBLKCP: no per-element issue slots); the < 16-byte
    // head and tail are plain loads
    const int mis = (int)(((uintptr_t)((p.lazy ? (const R*)p.vio : v) + base) & 15u) / sizeof(R));   // (a caller's vector need not be 16-byte aligned)
    R* const vs0 = S.vs + mis;                           // row 0 of the tile
    const unsigned char* vsm1 = (const unsigned char*)vs0 - 1;
    const int head = mis ? (RPV - mis < tlen ? RPV - mis : tlen) : 0;
    const int body = p.lazy ? 0 : ((tlen - head) / RPV) * RPV;
    if (p.lazy) {                                       // lazy normalisation: q_{j+1} formed while staging, written over y_j
      const R a = (R)p.st->a, ib = (R)p.st->inv_b;
      R* yq = p.vio + base;
      const R* qs = qprev + base;
      for (int x0 = tid; x0 < tlen; x0 += 8 * NT) {     // 16 loads in flight per thread before the first store
        R yv[8], qv[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int x = x0 + k * NT;
          yv[k] = x < tlen ? LDCS(&yq[x]) : (R)0;
          qv[k] = x < tlen ? LD_G(&qs[x]) : (R)0;
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int x = x0 + k * NT;
          if (x < tlen) {
            const R qn = (yv[k] - a * qv[k]) * ib;
            ST_S(&vs0[x], qn);
            ST_G(&yq[x], qn);
          }
        }
      }
    } else {                                            // stage the tile
      const R* src = v + base;
      if (body > 0 && tid == 0) {
        const uint32_t bytes = (uint32_t)body * (uint32_t)sizeof(R);
        mbar_arrive_expect_tx(&s_mbar, bytes);
        for (uint32_t o = 0; o < bytes; o += 32768u)      // 32 KB pieces
          bulk_copy_g2s((unsigned char*)(vs0 + head) + o, (const unsigned char*)(src + head) + o, bytes - o < 32768u ? bytes - o : 32768u, &s_mbar);
      }
      if (tid < head) ST_S(&vs0[tid], LD_G(&src[tid]));
      const int done = head + body;
      if (tid < tlen - done) ST_S(&vs0[done + tid], LD_G(&src[done + tid]));
    }
    const uint16_t* co = s_coloff + kT * nM;
    for (int M = tid; M < nM; M += NT) {                // column descriptors of this kT
      R coef = p.coef0;
      int n = 0;
      for (int e = 0; e < n_mm; ++e) {
        const uint32_t mk = p.mm_mask[e];
        if (__popc((uint32_t)M & mk) == 1) {
          MmEnt<R> me{};
          me.off = (uint32_t)LD_S(&co[(uint32_t)M ^ mk]); me.J = p.mm_J[e];
          ST_S(&S.dmm[M * n_mm + n], me);
          coef -= p.mm_J[e];
          ++n;
        }
      }
      ST_S(&S.dnmm[M], n);
      if (p.n_g) {                                       // left-over TT / TM bonds: rows of another tile, same lr
        int ng = 0;
        for (int g = 0; g < p.n_g; ++g) {
          const uint32_t tm = p.g_tmask[g];
          const int mb = p.g_mbit[g];
          bool act;
          int kTn = kT;
          uint32_t Mn = (uint32_t)M;
          if (mb < 0) { const uint32_t x = T & tm; act = x != 0 && x != tm; }
          else {
            const uint32_t tj = (T & tm) ? 1u : 0u, mi = ((uint32_t)M >> mb) & 1u;
            act = tj != mi;
            kTn = tj ? kT + 1 : kT - 1;                  // the one moves between T and the low part
            Mn = (uint32_t)M ^ (1u << mb);
          }
          if (act && kTn >= 0 && kTn <= p.mw) {
            const uint32_t Tn = T ^ tm;
            const uint64_t bn = p.mode == FTLM_INDEX_CLT ? passb_run_start<FTLM_INDEX_CLT>((uint64_t)Tn, p.mw, kTn, p.K, S.binom, p.clt)
                                                         : passb_run_start<FTLM_INDEX_CR>((uint64_t)Tn, p.mw, kTn, p.K, S.binom, p.clt);
            ST_S(&S.dg[M * p.n_g + ng], (uint32_t)(bn + LD_S(&s_coloff[kTn * nM + (int)Mn])));
            ST_S(&S.dgJ[M * p.n_g + ng], p.g_J[g]);
            coef -= p.g_J[g];
            ++ng;
          }
        }
        ST_S(&S.dng[M], ng);
      }
      ST_S(&S.dcoef[M], coef);
      for (int e = 0; e < n_ml; ++e) {
        const int j = p.ml_j[e];                         // padding entries: j = -1, never active (flo = 0, bit 31 = 0)
        ST_S(&S.dml[M * n_ml + e], j < 0 ? 0u : ((uint32_t)LD_S(&co[(uint32_t)M ^ (1u << j)]) * (uint32_t)sizeof(R) | (((uint32_t)M >> j) & 1u)));
      }
    }
#if !defined(FTLM_NEG_TEST) || FTLM_NEG_TEST != 3     // (negative test of the host emulation: tests/emu/build_emu.py)
    if (body > 0) { mbar_wait(&s_mbar, mbar_parity); mbar_parity ^= 1u; }   // the bulk copy has landed (every thread observes it)
#endif
    __syncthreads();                                    // descriptors, head and tail written by other threads
    // ---- units: one chunk of 32 low parts x a block of columns per warp ----------------------------
    const int u0 = LDG(&p.unit_off[kT]), u1 = LDG(&p.unit_off[kT + 1]);
    double s_qy = 0.0, s_yy = 0.0, s_qq = 0.0;
    (void)s_qy; (void)s_yy; (void)s_qq;
    for (int it = u0 + warp; it < u1; it += NW) {
      const uint32_t un = LDG(&p.units[it]);
      const int kL = (int)(un & 15u), chunk = (int)((un >> 4) & 15u), col0 = (int)((un >> 8) & 0xfffu), ncols = (int)(un >> 20);
      const int k0 = LD_S(&s_koff[kL]);
      const int len = LD_S(&s_koff[kL + 1]) - k0;
      const int lr = chunk * 32 + lane;
      const bool valid = lr < len;
      const int lrc = valid ? lr : 0;
      const int Lidx = k0 + lrc;
      uint32_t llo[NLL], flo[NML];                      // lane tables (registers)
#pragma unroll
      for (int e = 0; e < NLL; ++e) llo[e] = (uint32_t)LD_S(&s_ll[e * nL + Lidx]) * (uint32_t)sizeof(R);
#pragma unroll
      for (int e = 0; e < NML; ++e) {                    // byte offset of the flipped row | L_i
        const uint32_t f = (uint32_t)LD_S(&s_fl[e * nL + Lidx]);
        flo[e] = (f & 0x7fffu) * (uint32_t)sizeof(R) | (f >> 15);
      }
      const uint16_t* ml = s_mlist + LD_S(&s_moff[kT - kL]) + col0;
      uint32_t Mn = LD_S(&ml[0]);
      uint32_t cbn = LD_S(&co[Mn]);
      R qpn = (R)0;
      if (FUSED) qpn = LDCS(qprev + (base + cbn + (uint32_t)lrc));
      for (int c = 0; c < ncols; ++c) {
        const uint32_t M = Mn, cb = cbn;
        const R qp = qpn;
        if (c + 1 < ncols) {                              // q_prev of the next column is requested now
          Mn = LD_S(&ml[c + 1]);
          cbn = LD_S(&co[Mn]);
          if (FUSED) qpn = LDCS(qprev + (base + cbn + (uint32_t)lrc));
        }
        const unsigned char* colb = (const unsigned char*)(vs0 + cb);
        const R own = LD_S(&vs0[cb + (uint32_t)lrc]);
        // four independent partial sums (LL even/odd, ML even/odd) keep the FMA dependency chains short
        R acc = LD_S(&S.dcoef[M]) * own;
        R l0 = (R)0, l1 = (R)0, m0 = (R)0, m1 = (R)0;
        const uint32_t ownoff = (uint32_t)lrc * (uint32_t)sizeof(R);
#pragma unroll
        for (int e = 0; e < NLL; e += 2) {
          // a parallel bond's table entry is the row itself: only the antiparallel lanes read (fewer lanes per
          // shared-memory wavefront = fewer bank conflicts; emulated profile in profiles/r02_emu_smem_profile.md)
          const R a0 = LD_S_IF(llo[e] != ownoff, (const R*)(colb + llo[e]), own);
          const R a1 = LD_S_IF(llo[e + 1] != ownoff, (const R*)(colb + llo[e + 1]), own);
          if (UNIJ) { l0 += a0; l1 += a1; } else { l0 += p.ll_J[e] * a0; l1 += p.ll_J[e + 1] * a1; }
        }
        const int nmm = LD_S(&S.dnmm[M]);
        for (int a = 0; a < nmm; ++a) {
          const MmEnt<R> me = LD_S(&S.dmm[M * n_mm + a]);                  // one broadcast read: offset and J
          acc += me.J * LD_S(&vs0[me.off + (uint32_t)lrc]);
        }
        if (p.n_g) {
          const int ng = LD_S(&S.dng[M]);
          for (int a = 0; a < ng; ++a) acc += LD_S(&S.dgJ[M * p.n_g + a]) * LDG(v + ((size_t)LD_S(&S.dg[M * p.n_g + a]) + (uint32_t)lrc));
        }
#pragma unroll
        for (int e = 0; e < NML; e += 4) {                 // four column descriptors per 16-byte broadcast read
          const uint4 d4 = LD_S((const uint4*)&S.dml[M * n_ml + e]);
          const uint32_t d0 = d4.x, d1 = d4.y, d2 = d4.z, d3 = d4.w, f0 = flo[e], f1 = flo[e + 1], f2 = flo[e + 2], f3 = flo[e + 3];
          const R a0 = LD_S_IF((d0 ^ f0) & 1u, (const R*)(vsm1 + d0 + f0), own);   // active: exactly one of the two low bits is set
          const R a1 = LD_S_IF((d1 ^ f1) & 1u, (const R*)(vsm1 + d1 + f1), own);
          const R a2 = LD_S_IF((d2 ^ f2) & 1u, (const R*)(vsm1 + d2 + f2), own);
          const R a3 = LD_S_IF((d3 ^ f3) & 1u, (const R*)(vsm1 + d3 + f3), own);
          if (UNIJ) { m0 += a0; m1 += a1; m0 += a2; m1 += a3; }
          else { m0 += p.ml_J[e] * a0; m1 += p.ml_J[e + 1] * a1; m0 += p.ml_J[e + 2] * a2; m1 += p.ml_J[e + 3] * a3; }
        }
        if (UNIJ) acc += p.ll_J[0] * (l0 + l1) + p.ml_J[0] * (m0 + m1);
        else acc += (l0 + l1) + (m0 + m1);
        if (valid) {
          const uint64_t g = base + cb + (uint32_t)lrc;
          if (FUSED) {
            acc -= bprev * qp;
            if (FUSED == 1) {
              s_qy += (double)own * (double)acc;
              s_yy += (double)acc * (double)acc;
              s_qq += (double)own * (double)own;
            }
          }
          STCS(y + g, acc);
        }
      }
    }
    if (FUSED == 1) {                                   // deterministic per-tile partial sums
      const double a = warp_sum(s_qy), b = warp_sum(s_yy), c = warp_sum(s_qq);
      if (lane == 0) { ST_S(&S.red[warp * 3], a); ST_S(&S.red[warp * 3 + 1], b); ST_S(&S.red[warp * 3 + 2], c); }
      __syncthreads();
      if (tid < 3) {
        double s = 0.0;
        for (int wv = 0; wv < NW; ++wv) s += LD_S(&S.red[wv * 3 + tid]);
        ST_G(&p.partials[(size_t)tid * p.nT + T], s);
      }
    }
  }
  // ---- grid-wide finish: the last CTA resets the counters and (fused) advances the chain -----------
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
  double tot[3];
  for (int q = 0; q < 3; ++q) {                         // fixed assignment and order
    double a = 0.0;
    for (uint32_t k = tid; k < p.nT; k += NT) a += LD_G(&p.partials[(size_t)q * p.nT + k]);
    a = warp_sum(a);
    __syncthreads();
    if (lane == 0) ST_S(&S.red[warp], a);
    __syncthreads();
    double s = 0.0;
    if (tid == 0) for (int wv = 0; wv < NW; ++wv) s += LD_S(&S.red[wv]);
    tot[q] = s;
  }
  if (tid == 0) {
    ChainState* st = p.st;
    const double a = tot[0], b = tot[1], c = tot[2];
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

}  // namespace

// ---- host: plan, tables, launch -------------------------------------------------------------------
namespace {

uint64_t binom_r(int n, int k) {
  if (k < 0 || k > n) return 0;
  if (k > n - k) k = n - k;
  unsigned __int128 r = 1;
  for (int i = 1; i <= k; ++i) r = r * (unsigned)(n - k + i) / (unsigned)i;
  return (uint64_t)r;
}

template <typename R>
size_t tmlr_smem_bytes(const ftlm_ctx* c, const TmlrPlan* t) {
  TmlrSmem<R> S;
  return tmlr_layout<R>(S, nullptr, c->N, c->N_up, t->blob_bytes, t->max_tile, 1 << t->m, t->n_mm, t->n_ml, t->n_g, TMLR_THREADS / 32);
}

template <typename R, int NLL, int NML>
int launch_tmlr_k(ftlm_ctx* c, const TmlrParams<R>& p, int grid, size_t smem, const void* v, const void* qp, void* y, cudaStream_t s) {
  if (c->tmlr->unij) {
    auto k = hv_tmlr_kernel<R, NLL, NML, true>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    FTLM_LAUNCH(k, grid, TMLR_THREADS, smem, s, p, (const R*)v, (const R*)qp, (R*)y);
  } else {
    auto k = hv_tmlr_kernel<R, NLL, NML, false>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    FTLM_LAUNCH(k, grid, TMLR_THREADS, smem, s, p, (const R*)v, (const R*)qp, (R*)y);
  }
  CK(cudaGetLastError());
  return FTLM_OK;
}

template <typename R, int NLL>
int launch_tmlr_ml(ftlm_ctx* c, const TmlrParams<R>& p, int grid, size_t smem, const void* v, const void* qp, void* y, cudaStream_t s) {
  switch (p.n_ml) {
    case 4: return launch_tmlr_k<R, NLL, 4>(c, p, grid, smem, v, qp, y, s);
    case 8: return launch_tmlr_k<R, NLL, 8>(c, p, grid, smem, v, qp, y, s);
    case 12: return launch_tmlr_k<R, NLL, 12>(c, p, grid, smem, v, qp, y, s);
    default: return launch_tmlr_k<R, NLL, 16>(c, p, grid, smem, v, qp, y, s);
  }
}

template <typename R>
int launch_tmlr(ftlm_ctx* c, const void* v, const void* qp, void* y, int fused, cudaStream_t s, void* vio = nullptr) {
  TmlrPlan* t = c->tmlr;
  TmlrParams<R> p;
  memset(&p, 0, sizeof(p));
  p.N = c->N; p.K = c->N_up; p.w = t->w; p.m = t->m; p.mw = t->w + t->m;
  p.nT = t->nT; p.t_begin = 0; p.t_end = t->nT;
  if (c->debug_item_count > 0) {
    p.t_begin = (uint32_t)std::min<int64_t>(c->debug_item_first, t->nT);
    p.t_end = (uint32_t)std::min<int64_t>(c->debug_item_first + c->debug_item_count, t->nT);
  }
  p.n_ll = t->n_ll; p.n_mm = t->n_mm; p.n_ml = t->n_ml; p.max_tile = t->max_tile;
  p.mode = c->mode; p.fused = fused;
  p.lazy = vio ? 1 : 0; p.vio = (R*)vio;
  p.dim = c->dim; p.binom = c->d_binom64; p.clt = c->d_clt; p.blob = t->d_blob; p.blob_bytes = t->blob_bytes;
  p.off_koff = t->off_koff; p.off_tlen = t->off_tlen; p.off_coloff = t->off_coloff; p.off_mlist = t->off_mlist;
  p.off_moff = t->off_moff; p.off_ll = t->off_ll; p.off_fl = t->off_fl;
  p.units = t->d_units; p.unit_off = t->d_unit_off; p.partials = t->d_partials; p.counter = t->d_counter;
  p.st = c->d_state; p.coef0 = (R)t->coef0;
  for (int e = 0; e < t->n_ll; ++e) p.ll_J[e] = (R)t->ll_J[(size_t)e];
  for (int e = 0; e < t->n_ml; ++e) { p.ml_J[e] = (R)t->ml_J[(size_t)e]; p.ml_j[e] = t->ml_j[(size_t)e]; }
  for (int e = 0; e < t->n_mm; ++e) { p.mm_J[e] = (R)t->mm_J[(size_t)e]; p.mm_mask[e] = t->mm_mask[(size_t)e]; }
  p.n_g = t->n_g;
  for (int g = 0; g < t->n_g; ++g) { p.g_tmask[g] = t->g_tmask[(size_t)g]; p.g_mbit[g] = t->g_mbit[(size_t)g]; p.g_J[g] = (R)t->g_J[(size_t)g]; }
  int grid = c->sm_count;
  if ((uint32_t)grid > p.t_end - p.t_begin) grid = (int)std::max(1u, p.t_end - p.t_begin);
  const size_t smem = tmlr_smem_bytes<R>(c, t);
  switch (p.n_ll) {
    case 4: return launch_tmlr_ml<R, 4>(c, p, grid, smem, v, qp, y, s);
    case 8: return launch_tmlr_ml<R, 8>(c, p, grid, smem, v, qp, y, s);
    case 12: return launch_tmlr_ml<R, 12>(c, p, grid, smem, v, qp, y, s);
    default: return launch_tmlr_ml<R, 16>(c, p, grid, smem, v, qp, y, s);
  }
}

}  // namespace

void ftlm_tmlr_plan_destroy(ftlm_ctx* c) {
  TmlrPlan* t = c->tmlr;
  if (!t) return;
  ftlm_dfree(t->d_blob); ftlm_dfree(t->d_units); ftlm_dfree(t->d_unit_off); ftlm_dfree(t->d_partials); ftlm_dfree(t->d_counter);
  delete t;
  c->tmlr = nullptr;
}

// Build the plan for the split (w, m).  in_window[b] != 0: bond b belongs to a PASS-B window.  Leaves
// c->tmlr == nullptr (FTLM_OK) when the kernel cannot serve this sector: a bond outside the windows
// leaves the tile, a bond class overflows the register tables, or the tables do not fit shared memory.
int ftlm_tmlr_plan_create(ftlm_ctx* c, int w, int m, const std::vector<int>& in_window) {
  ftlm_tmlr_plan_destroy(c);
  const int N = c->N, mw = w + m, t = N - mw;
  if (w < 5 || w > 11 || m < 1 || m > 12 || t < 1 || t > 22 || c->dim < 64 || (uint64_t)c->dim >= (1ull << 32)) return FTLM_OK;
  TmlrPlan* P = new TmlrPlan();
  P->w = w; P->m = m; P->nT = 1u << t;
  struct LLb { uint32_t mask; };
  struct MLb { int i, j; };
  std::vector<LLb> ll;
  std::vector<MLb> mlb;
  double sumJ = 0.0;
  for (int b = 0; b < c->nb; ++b) {
    if (in_window[(size_t)b]) continue;
    const BondDev& d = c->bonds[(size_t)b];
    if (d.j >= mw) {                                                    // leaves the tile and no window took it
      if (d.i < w || (int)P->g_tmask.size() >= TMLR_MAX_G) { delete P; return FTLM_OK; }   // TL: per-lane global gather, not served here
      P->g_tmask.push_back((uint32_t)(d.mask >> mw));                   // TT: both bits; TM: the T bit (the M bit shifts out)
      P->g_mbit.push_back(d.i >= mw ? -1 : d.i - w);
      P->g_J.push_back(d.Jh);
      continue;
    }
    if (d.j < w) { ll.push_back({(uint32_t)d.mask}); P->ll_J.push_back(d.Jh); sumJ += d.Jh; }
    else if (d.i >= w) { P->mm_mask.push_back((uint32_t)(d.mask >> w)); P->mm_J.push_back(d.Jh); }
    else { mlb.push_back({d.i, d.j - w}); P->ml_J.push_back(d.Jh); P->ml_j.push_back(d.j - w); sumJ += d.Jh; }
  }
  if (ll.size() > TMLR_MAX_LL || P->mm_mask.size() > TMLR_MAX_MM || mlb.size() > TMLR_MAX_ML) { delete P; return FTLM_OK; }
  // uniform couplings (and at least one bond in each list): the kernel adds first and multiplies once
  P->unij = !ll.empty() && !mlb.empty() && c->unij_allowed;
  for (size_t e = 1; e < P->ll_J.size(); ++e) P->unij = P->unij && P->ll_J[e] == P->ll_J[0];
  for (size_t e = 1; e < P->ml_J.size(); ++e) P->unij = P->unij && P->ml_J[e] == P->ml_J[0];
  // pad the LL / ML lists to multiples of 4 (at least 4): LL target = the row itself, ML never active (reads the
  // row itself); J = 0, or - uniform case - the common J with the added J * v_t taken back from the diagonal
  while (ll.size() < 4 || (ll.size() & 3)) {
    ll.push_back({0u});
    if (P->unij) { P->ll_J.push_back(P->ll_J[0]); sumJ += P->ll_J[0]; } else P->ll_J.push_back(0.0);
  }
  while (mlb.size() < 4 || (mlb.size() & 3)) {
    mlb.push_back({-1, -1});
    P->ml_j.push_back(-1);
    if (P->unij) { P->ml_J.push_back(P->ml_J[0]); sumJ += P->ml_J[0]; } else P->ml_J.push_back(0.0);
  }
  P->n_ll = (int)ll.size(); P->n_mm = (int)P->mm_mask.size(); P->n_ml = (int)mlb.size(); P->n_g = (int)P->g_tmask.size();
  P->max_tile = (int)binom_r(mw, mw / 2);
  if (P->max_tile > 65535) { delete P; return FTLM_OK; }
  P->coef0 = c->diag0 - sumJ;
  const int nL = 1 << w, nM = 1 << m;
  std::vector<int> koff((size_t)w + 2, 0);
  for (int k = 0; k <= w; ++k) koff[(size_t)k + 1] = koff[(size_t)k] + (int)binom_r(w, k);
  std::vector<uint16_t> lr((size_t)nL), lstate((size_t)nL);
  for (int L = 0; L < nL; ++L) {                                          // lr(L): rank among the w-bit words of equal popcount
    uint64_t r = 0;
    int cnt = 0;
    for (int q = 0; q < w; ++q)
      if ((L >> q) & 1) { ++cnt; r += binom_r(q, cnt); }
    lr[(size_t)L] = (uint16_t)r;
    lstate[(size_t)(koff[(size_t)cnt] + (int)r)] = (uint16_t)L;
  }
  std::vector<uint16_t> mlist((size_t)nM);
  std::vector<int> moff((size_t)m + 2, 0);
  for (int k = 0; k <= m; ++k) moff[(size_t)k + 1] = moff[(size_t)k] + (int)binom_r(m, k);
  {
    std::vector<int> fill(moff.begin(), moff.end() - 1);
    for (int M = 0; M < nM; ++M) mlist[(size_t)fill[(size_t)__builtin_popcount((unsigned)M)]++] = (uint16_t)M;
  }
  std::vector<int> tlen((size_t)mw + 1);
  std::vector<uint16_t> coloff((size_t)(mw + 1) * nM, 0);
  std::vector<uint32_t> units;
  std::vector<int> unit_off((size_t)mw + 2, 0);
  for (int kT = 0; kT <= mw; ++kT) {
    tlen[(size_t)kT] = (int)binom_r(mw, kT);
    int off = 0;
    for (int M = 0; M < nM; ++M) {
      coloff[(size_t)kT * nM + M] = (uint16_t)off;
      const int kL = kT - __builtin_popcount((unsigned)M);
      if (kL >= 0 && kL <= w) off += (int)binom_r(w, kL);
    }
    // units: (kL, chunk of 32 low parts) x blocks of CB columns; CB sized so that a tile has ~6 units per warp
    long total = 0;
    for (int kL = std::max(0, kT - m); kL <= std::min(w, kT); ++kL) total += (long)((binom_r(w, kL) + 31) / 32) * (long)binom_r(m, kT - kL);
    const int CB = (int)std::max<long>(4, std::min<long>(64, total / (6 * (TMLR_THREADS / 32))));
    const size_t first = units.size();
    for (int kL = std::max(0, kT - m); kL <= std::min(w, kT); ++kL) {
      const int nch = (int)((binom_r(w, kL) + 31) / 32), ncol = (int)binom_r(m, kT - kL);
      for (int ch = 0; ch < nch; ++ch)
        for (int c0 = 0; c0 < ncol; c0 += CB)
          units.push_back((uint32_t)kL | ((uint32_t)ch << 4) | ((uint32_t)c0 << 8) | ((uint32_t)std::min(CB, ncol - c0) << 20));
    }
    std::stable_sort(units.begin() + (long)first, units.end(), [](uint32_t a, uint32_t b) { return (a >> 20) > (b >> 20); });
    unit_off[(size_t)kT + 1] = (int)units.size();
  }
  std::vector<uint16_t> lltab((size_t)std::max(P->n_ll, 1) * nL, 0), fltab((size_t)std::max(P->n_ml, 1) * nL, 0);
  for (int k = 0; k <= w; ++k)
    for (int r = 0; r < koff[(size_t)k + 1] - koff[(size_t)k]; ++r) {
      const int Lidx = koff[(size_t)k] + r;
      const uint32_t L = lstate[(size_t)Lidx];
      for (int e = 0; e < P->n_ll; ++e) {
        const uint32_t mk = ll[(size_t)e].mask, x = L & mk;
        lltab[(size_t)e * nL + Lidx] = (uint16_t)((x != 0 && x != mk) ? lr[(size_t)(L ^ mk)] : (uint32_t)r);   // parallel: the row itself
      }
      for (int e = 0; e < P->n_ml; ++e) {
        const int i = mlb[(size_t)e].i;
        if (i < 0) continue;                                              // padding: 0 (bit 15 clear, never active)
        fltab[(size_t)e * nL + Lidx] = (uint16_t)((uint32_t)lr[(size_t)(L ^ (1u << i))] | (((L >> i) & 1u) << 15));
      }
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
  P->off_mlist = put(mlist.data(), mlist.size() * 2);
  P->off_moff = put(moff.data(), moff.size() * 4);
  P->off_ll = put(lltab.data(), lltab.size() * 2);
  P->off_fl = put(fltab.data(), fltab.size() * 2);
  P->blob_bytes = (int)blob.size();
  c->tmlr = P;
  P->smem = c->prec == FTLM_FP32 ? tmlr_smem_bytes<float>(c, P) : tmlr_smem_bytes<double>(c, P);
  if (P->smem > (size_t)227 * 1024 - 1024) { c->tmlr = nullptr; delete P; return FTLM_OK; }
  auto up = [&](void** d, const void* h, size_t bytes) -> bool {
    if (ftlm_dmalloc(d, bytes ? bytes : 16) != cudaSuccess) return false;
    if (bytes && h && cudaMemcpy(*d, h, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return false;
    return true;
  };
  const size_t pbytes = (size_t)P->nT * 24;
  bool ok = up((void**)&P->d_blob, blob.data(), blob.size()) && up((void**)&P->d_units, units.data(), units.size() * 4) &&
            up((void**)&P->d_unit_off, unit_off.data(), unit_off.size() * 4) &&
            up((void**)&P->d_partials, nullptr, pbytes) && up((void**)&P->d_counter, nullptr, 16);
  if (ok) ok = cudaMemset(P->d_partials, 0, pbytes) == cudaSuccess && cudaMemset(P->d_counter, 0, 16) == cudaSuccess;
  if (!ok) { cudaGetLastError(); ftlm_tmlr_plan_destroy(c); ftlm_set_error("TMLR: table upload failed"); return FTLM_ENOMEM; }
  return FTLM_OK;
}

int64_t ftlm_tmlr_info(const ftlm_ctx* c, const char* key) {
  const TmlrPlan* t = c->tmlr;
  if (!strcmp(key, "tmlr_available")) return t ? 1 : 0;
  if (!t) return -1;
  if (!strcmp(key, "tmlr_smem")) return (int64_t)t->smem;
  if (!strcmp(key, "tmlr_unij_used")) return t->unij ? 1 : 0;
  if (!strcmp(key, "tmlr_n_ll")) return t->n_ll;
  if (!strcmp(key, "tmlr_n_mm")) return t->n_mm;
  if (!strcmp(key, "tmlr_n_ml")) return t->n_ml;
  if (!strcmp(key, "tmlr_n_g")) return t->n_g;
  return -1;
}

int ftlm_launch_hv_tmlr(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, cudaStream_t s) {
  if (!c->tmlr) { ftlm_set_error("TMLR kernel unavailable"); return FTLM_EUNSUPPORTED; }
  if (c->prec == FTLM_FP32) return launch_tmlr<float>(c, v, qprev, y, fused, s);
  return launch_tmlr<double>(c, v, qprev, y, fused, s);
}

bool ftlm_tmlr_lazy_ok(const ftlm_ctx* c) { return c->use_tmlr && c->tmlr && c->tmlr->n_g == 0; }

int ftlm_launch_hv_tmlr_lazy(ftlm_ctx* c, void* yq, const void* q, void* y, int fused, cudaStream_t s) {
  if (!ftlm_tmlr_lazy_ok(c) || !fused) { ftlm_set_error("TMLR lazy pass unavailable"); return FTLM_EUNSUPPORTED; }
  // v is only read through vio in this form (n_g == 0: no reads of other tiles); q is q_j = this step's q_prev
  if (c->prec == FTLM_FP32) return launch_tmlr<float>(c, yq, q, y, fused, s, yq);
  return launch_tmlr<double>(c, yq, q, y, fused, s, yq);
}
