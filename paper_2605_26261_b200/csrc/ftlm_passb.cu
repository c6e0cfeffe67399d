// PASS-B kernels - bonds among the top label bits, streamed.
//
// For a bond whose two sites lie in a window S = [lo, lo+s) of high label positions the swap
// P_b (Eq. 12-14 at s = 1/2: y_t += (J_b/2)(v[P_b n_t] - v[n_t])) maps the contiguous run of rows
// (F, u, *) onto the run (F, u', *), u' = u with the two window bits exchanged, element by element
// (same low part, same offset x inside the run).  One work item = one (F, popc(u)) class and one
// chunk of X = 32 k run offsets:
//   phase 1: the C(s, p_S) run chunks v[start(F,u) + x0 .. + X) are loaded into shared memory,
//            tile[slot(u) * X + x]  (coalesced, every element of v read once per window);
//   phase 2: one warp per u adds, for its X rows, sum_b (J_b/2) (tile[slot(u'_b)][x] - tile[slot(u)][x])
//            to y (coalesced read-modify-write).  The antiparallel bonds of u and the slots of the
//            u'_b come from a precomputed row of 32 entries per u (one coalesced load, then
//            warp-broadcast), so the inner loop is one shuffle, one shared-memory read and one FMA.
// Run starts are sector indices of the first label of a run, by CR or CLT (ftlm_passb.cuh).
// The last window carries the fused Lanczos reductions (it writes the final y): per-item FP64
// partial sums in a buffer indexed by item, added in fixed order by the last CTA (bit-reproducible).
#include <algorithm>
#include <cstring>
#include <vector>

#define FTLM_TU 5
#include "ftlm_passb.cuh"
#include "ftlm_vec.cuh"

#define PASSB_MAX_BONDS 28          // neighbour rows of 32 entries: up to 28 bonds (padded to multiples of 4), entry 31 holds the count and the sum of J
#define PASSB_MAX_S 12
#define PASSB_THREADS 1024
#define PASSB_END 0xFFFFFFFFu
#define PASSB_XK 2                  // run offsets per lane and window word (X = 32 * xk, xk <= PASSB_XK)
#define PASSB_RED_DOUBLES (32 * 3 * FTLM_MAX_BATCH + 64 + 3 * FTLM_MAX_BATCH + 4)   // per-warp sums + finish_chains scratch; even: the tile behind it stays 16-byte aligned
#define PASSB_PF 8                  // window words whose y is in flight per warp (divided by the batch: registers)

template <typename R>
struct PassBParams {
  int N, K, lo, s, f, ngroups;
  uint32_t nitems;
  uint32_t item_begin, item_end;    // items handed out: [item_begin, item_end)  (all unless option "debug_items")
  uint64_t smask_hi, fmask_hi;      // active / frozen positions of the label >> lo
  int64_t dim;
  const uint64_t* binom;            // [(N+1)*(K+1)] global
  const uint2* clt;
  const uint16_t* ustate;           // [2^s]: window words grouped by popcount, ascending inside a group
  const int* koff;                  // [s+2]: first slot of popcount class p in ustate
  const uint32_t* nbr_off;          // [2^s][32], row = position of u in ustate: index of row slot(u') * X in the tile; [31] = number of entries
  const R* nbr_J;                   // [2^s][32]: J_b/2 of the same entries; [31] = their sum
  const uint32_t* grp_first;        // [ngroups+1]: first item of group g = F*(s+1) + p_S
  const uint32_t* item_group;       // [nitems]: group of every item
  double* partials;                 // [3 * B][nitems]
  unsigned int* counter;            // [0] item counter, [1] ticket
  ChainState* st;                   // [B]
  int xk[PASSB_MAX_S + 1];          // X/32 per popcount class
  int max_conf;                     // largest C(s, p_S) among non-empty classes
  int unij;                         // every bond of the window has the same J_b/2 (= Juni)
  R Juni;
};

struct PassBWindow {
  int lo = 0, s = 0, f = 0, ngroups = 0, max_conf = 0;
  uint64_t smask = 0;               // the s active label positions (all >= lo)
  int ctas = 1, threads = PASSB_THREADS;
  uint32_t nitems = 0;
  int xk[PASSB_MAX_S + 1] = {0};
  size_t smem = 0;
  std::vector<int> bonds;           // indices into ctx->bonds
  std::vector<double> Jh;
  uint16_t* d_ustate = nullptr;
  int* d_koff = nullptr;
  uint32_t* d_nbr = nullptr;          // row indices in the tile
  void* d_nbrJ = nullptr;             // J_b/2 in the handle's precision
  uint32_t* d_grp_first = nullptr;
  uint32_t* d_item_group = nullptr;
  double* d_partials = nullptr;
  unsigned int* d_counter = nullptr;
};

struct PassBSet {
  std::vector<PassBWindow> win;
};

namespace {

__host__ __device__ inline uint64_t bits_deposit(uint64_t x, uint64_t mask) {
  uint64_t r = 0;
  for (int k = 0; mask; ++k) {
    const uint64_t low = mask & (~mask + 1ull);
    if ((x >> k) & 1ull) r |= low;
    mask ^= low;
  }
  return r;
}

// esz = bytes of one row of the batch (element size x chains)
__host__ __device__ inline size_t passb_smem_bytes(int N, int K, int max_conf, int max_rows, int esz) {
  size_t o = 0;
  o += ((size_t)(N + 1) * (K + 1) * 8 + 15) & ~(size_t)15;      // binom
  o += ((size_t)max_conf * 8 + 15) & ~(size_t)15;               // run starts
  o += (size_t)PASSB_RED_DOUBLES * 8;                           // reduction scratch (per-warp sums; finish_chains)
  o += (size_t)max_rows * esz;                                  // tile: max over classes of C(s,p) * X
  return o;
}

// Phase 2 of one work item, specialised on the run offsets per lane (XKC), on uniform couplings (UNIJ) and on the
// batch B (rows of B interleaved chains, L207) so that an item executes one straight variant of the word loop.
template <typename R, int B, bool FUSED, int XKC, bool UNIJ>
__device__ __forceinline__ void passb_phase2(const PassBParams<R>& p, const Vec<R, B>* tile, Vec<R, B>* __restrict__ y, const uint64_t* s_start,
                                             int c0, int nconf, int X, uint64_t x0, int nx, int lane, int warp, int NW,
                                             double* s_qy, double* s_yy, double* s_qq) {
  typedef Vec<R, B> V;
  constexpr int PF = PASSB_PF / B;
  for (int sl0 = warp; sl0 < nconf; sl0 += NW * PF) {
    V yold[PF][PASSB_XK];
    uint64_t rstart[PF];                               // run start of each word: read once from shared memory
#pragma unroll
    for (int j = 0; j < PF; ++j) {
      const int sl = sl0 + j * NW;
      rstart[j] = sl < nconf ? LD_S(&s_start[sl]) : 0ull;
#pragma unroll
      for (int k = 0; k < PASSB_XK; ++k) {
        const int x = lane + 32 * k;
        if (sl < nconf && k < XKC && x < nx) yold[j][k] = vec_ldcs(y + rstart[j] + x0 + x);
        else yold[j][k] = V{};
      }
    }
#pragma unroll
    for (int j = 0; j < PF; ++j) {
      const int sl = sl0 + j * NW;
      if (sl >= nconf) break;
      // the word's neighbour row: entries 0 .. cnt-1 (cnt a multiple of 4: padded with the word's own tile row and
      // J = 0), entry 31 = cnt / sum of J.  Every lane reads the same addresses: 16-byte broadcast loads that stay in
      // L1 (one load per four bonds instead of one shuffle per bond).
      const uint32_t* nro = p.nbr_off + (size_t)(c0 + sl) * 32;
      const R* nrJ = p.nbr_J + (size_t)(c0 + sl) * 32;
      const int cnt = (int)LDG(&nro[31]);
      const R sumJ = LDG(&nrJ[31]);
      // lanes past the end of the run (x >= nx) read stale tile words and are discarded at the store
      const unsigned char* tl = (const unsigned char*)tile + (size_t)lane * sizeof(V);
      V* yrow = y + rstart[j] + x0;
      V own[PASSB_XK], acc[PASSB_XK];
      own[0] = LD_S((const V*)(tl + (size_t)sl * X * sizeof(V)));
      acc[0] = V{};
      own[1] = V{}; acc[1] = V{};
      if (XKC == 2) own[1] = LD_S((const V*)(tl + (size_t)sl * X * sizeof(V) + 32 * sizeof(V)));
#pragma unroll 2
      for (int e = 0; e < cnt; e += 4) {
        const uint4 o4 = LDG((const uint4*)(nro + e));
        const uint32_t oo[4] = {o4.x, o4.y, o4.z, o4.w};
        R jj[4];
        if (!UNIJ) {
          if constexpr (sizeof(R) == 4) { const uint4 j4 = LDG((const uint4*)(nrJ + e)); jj[0] = __uint_as_float(j4.x); jj[1] = __uint_as_float(j4.y); jj[2] = __uint_as_float(j4.z); jj[3] = __uint_as_float(j4.w); }
          else { const double2 ja = LDG((const double2*)(nrJ + e)), jb = LDG((const double2*)(nrJ + e + 2)); jj[0] = (R)ja.x; jj[1] = (R)ja.y; jj[2] = (R)jb.x; jj[3] = (R)jb.y; }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const unsigned char* src = tl + (size_t)oo[q] * sizeof(V);       // row index -> byte offset
          const V g0 = LD_S((const V*)src);
          V g1 = V{};
          if (XKC == 2) g1 = LD_S((const V*)(src + 32 * sizeof(V)));
#pragma unroll
          for (int c = 0; c < B; ++c) {
            if (UNIJ) { acc[0].x[c] += g0.x[c]; if (XKC == 2) acc[1].x[c] += g1.x[c]; }
            else { acc[0].x[c] += jj[q] * g0.x[c]; if (XKC == 2) acc[1].x[c] += jj[q] * g1.x[c]; }
          }
        }
      }
      if (UNIJ) {
#pragma unroll
        for (int c = 0; c < B; ++c) { acc[0].x[c] *= p.Juni; acc[1].x[c] *= p.Juni; }
      }
#pragma unroll
      for (int k = 0; k < PASSB_XK; ++k) {
        const int x = lane + 32 * k;
        if (k < XKC && x < nx) {
          V yn;
#pragma unroll
          for (int c = 0; c < B; ++c) {
            yn.x[c] = yold[j][k].x[c] + (acc[k].x[c] - sumJ * own[k].x[c]);
            if (FUSED) {
              s_qy[c] += (double)own[k].x[c] * (double)yn.x[c];
              s_yy[c] += (double)yn.x[c] * (double)yn.x[c];
              s_qq[c] += (double)own[k].x[c] * (double)own[k].x[c];
            }
          }
          vec_stcs(&yrow[x], yn);
        }
      }
    }
  }
}

// rows wider than 4 bytes (FP64, batches) run with 512 threads per CTA: 128 registers per thread instead of 64
// (ptxas: the y prefetch of 8 / B window words x 2 offsets spills at 64)
template <typename R, int B, int MODE, bool FUSED>
__global__ void __launch_bounds__((sizeof(R) * B > 4) ? 512 : PASSB_THREADS, 1)
passb_kernel(const __grid_constant__ PassBParams<R> p, const R* __restrict__ v_, R* __restrict__ y_) {
  typedef Vec<R, B> V;
  FTLM_DYN_SMEM(smem);
  __shared__ unsigned int s_item;
  __shared__ bool s_last;
  if (FUSED) {
    bool all_done = true;
#pragma unroll
    for (int c = 0; c < B; ++c) all_done = all_done && p.st[c].done;
    if (all_done) return;
  }
  const V* __restrict__ v = (const V*)v_;
  V* __restrict__ y = (V*)y_;
  const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
  const int K1 = p.K + 1;
  uint64_t* s_binom = (uint64_t*)smem;
  size_t o = ((size_t)(p.N + 1) * K1 * 8 + 15) & ~(size_t)15;
  uint64_t* s_start = (uint64_t*)(smem + o);
  o += ((size_t)p.max_conf * 8 + 15) & ~(size_t)15;
  double* s_red = (double*)(smem + o);
  o += (size_t)PASSB_RED_DOUBLES * 8;
  static_assert((PASSB_RED_DOUBLES * 8) % 16 == 0, "tile alignment");
  V* tile = (V*)(smem + o);
  for (int k = tid; k < (p.N + 1) * K1; k += NT) ST_S(&s_binom[k], LD_G(&p.binom[k]));
  int cur_group = -1;
  const int s1 = p.s + 1;

  if (tid == 0) s_item = atomicAdd(&p.counter[0], 1u);
  for (;;) {
    __syncthreads();                                   // previous item done (tile, starts reusable), next item id visible
    const uint32_t item = s_item + p.item_begin;
    __syncthreads();                                   // everyone has read it
    if (item >= p.item_end) break;
    if (tid == 0) s_item = atomicAdd(&p.counter[0], 1u);   // the following item's id travels while this item is processed
    const int g = (int)LDG(&p.item_group[item]);      // group g = F * (s+1) + p_S of this item
    const uint32_t F = (uint32_t)(g / s1);
    const int pS = g - (int)F * s1;
    const int kP = p.K - __popc(F) - pS;                // in [0, lo] by construction of the groups
    const int c0 = LDG(&p.koff[pS]);
    const int nconf = LDG(&p.koff[pS + 1]) - c0;
    const int XK = p.xk[pS];
    const int X = 32 * XK;
    const uint64_t RL = LD_S(&s_binom[p.lo * K1 + kP]);        // run length C(lo, kP)
    const uint64_t x0 = (uint64_t)(item - LDG(&p.grp_first[g])) * (uint64_t)X;
    if (g != cur_group) {                               // (uniform) run starts of this class
      for (int sl = tid; sl < nconf; sl += NT) {
        const uint64_t hi = bits_deposit((uint64_t)F, p.fmask_hi) | bits_deposit((uint64_t)LDG(&p.ustate[c0 + sl]), p.smask_hi);
        ST_S(&s_start[sl], passb_run_start<MODE>(hi, p.lo, kP, p.K, s_binom, p.clt));
      }
      cur_group = g;
      __syncthreads();
    }
    const uint64_t left = RL - x0;                      // rows of the run at or after x0 (> 0)
    const int nx = left < (uint64_t)X ? (int)left : X;  // valid offsets in this chunk
    // ---- phase 1: stage the run chunks (cp.async: every copy of the item is in flight at once) ------
    for (int sl = warp; sl < nconf; sl += NW) {
      const V* src = v + LD_S(&s_start[sl]) + x0;
      V* dst = tile + (size_t)sl * X;
#pragma unroll
      for (int k = 0; k < PASSB_XK; ++k) {
        const int x = lane + 32 * k;
        if (k < XK && x < nx) cp_async_vec(&dst[x], &src[x]);
      }
    }
#if !defined(FTLM_NEG_TEST) || FTLM_NEG_TEST != 1     // (negative test of the host emulation: tests/emu/build_emu.py)
    cp_async_wait_all();
#endif
    __syncthreads();
    // ---- phase 2: one warp per window word; y of PASSB_PF / B words is requested before the first is used ---
    double s_qy[B], s_yy[B], s_qq[B];
#pragma unroll
    for (int c = 0; c < B; ++c) { s_qy[c] = 0.0; s_yy[c] = 0.0; s_qq[c] = 0.0; }
    if (XK == 1) {
      if (p.unij) passb_phase2<R, B, FUSED, 1, true>(p, tile, y, s_start, c0, nconf, X, x0, nx, lane, warp, NW, s_qy, s_yy, s_qq);
      else passb_phase2<R, B, FUSED, 1, false>(p, tile, y, s_start, c0, nconf, X, x0, nx, lane, warp, NW, s_qy, s_yy, s_qq);
    } else {
      if (p.unij) passb_phase2<R, B, FUSED, 2, true>(p, tile, y, s_start, c0, nconf, X, x0, nx, lane, warp, NW, s_qy, s_yy, s_qq);
      else passb_phase2<R, B, FUSED, 2, false>(p, tile, y, s_start, c0, nconf, X, x0, nx, lane, warp, NW, s_qy, s_yy, s_qq);
    }
    if (FUSED) {                                        // deterministic per-item partial sums
#pragma unroll
      for (int c = 0; c < B; ++c) {
        const double a = warp_sum(s_qy[c]), b = warp_sum(s_yy[c]), cc = warp_sum(s_qq[c]);
        if (lane == 0) { ST_S(&s_red[warp * 3 * B + 3 * c], a); ST_S(&s_red[warp * 3 * B + 3 * c + 1], b); ST_S(&s_red[warp * 3 * B + 3 * c + 2], cc); }
      }
      __syncthreads();
      if (tid < 3 * B) {
        double s = 0.0;
        for (int wv = 0; wv < NW; ++wv) s += LD_S(&s_red[wv * 3 * B + tid]);
        ST_G(&p.partials[(size_t)tid * p.nitems + item], s);
      }
    }
  }
  // ---- grid-wide finish: the last CTA resets the counters and (fused) advances the chains ---------
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_last = (atomicAdd(&p.counter[1], 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (tid == 0) { p.counter[0] = 0; p.counter[1] = 0; }
  if (!FUSED) return;
  finish_chains<B>(p.partials, p.nitems, p.st, s_red + 32 * 3 * FTLM_MAX_BATCH);
}

// bit k of x goes to the position of the k-th set bit of mask / back
__host__ __device__ inline uint64_t bits_extract(uint64_t x, uint64_t mask) {
  uint64_t r = 0;
  for (int k = 0; mask; ++k) {
    const uint64_t low = mask & (~mask + 1ull);
    if (x & low) r |= 1ull << k;
    mask ^= low;
  }
  return r;
}

uint64_t binom_b(int n, int k) {
  if (k < 0 || k > n) return 0;
  if (k > n - k) k = n - k;
  unsigned __int128 r = 1;
  for (int i = 1; i <= k; ++i) r = r * (unsigned)(n - k + i) / (unsigned)i;
  return (uint64_t)r;
}

}  // namespace

// ---- host: window selection, tables, launch -----------------------------------------------------
void ftlm_passb_plan_destroy(ftlm_ctx* c) {
  PassBSet* S = c->passb;
  if (!S) return;
  for (PassBWindow& w : S->win) {
    ftlm_dfree(w.d_ustate); ftlm_dfree(w.d_koff); ftlm_dfree(w.d_nbr); ftlm_dfree(w.d_nbrJ); ftlm_dfree(w.d_grp_first); ftlm_dfree(w.d_item_group);
    ftlm_dfree(w.d_partials); ftlm_dfree(w.d_counter);
  }
  delete S;
  c->passb = nullptr;
}

int ftlm_passb_windows(const ftlm_ctx* c) { return c->passb ? (int)c->passb->win.size() : 0; }

void ftlm_passb_window_geometry(const ftlm_ctx* c, int window, int* lo, int* s) {
  const PassBWindow& w = c->passb->win[(size_t)window];
  *lo = w.lo; *s = w.s;
}

int64_t ftlm_passb_info(const ftlm_ctx* c, const char* key) {
  const PassBSet* S = c->passb;
  if (!strcmp(key, "passb_windows")) return S ? (int64_t)S->win.size() : 0;
  if (!S || S->win.empty()) return -1;
  if (!strcmp(key, "passb_bonds")) { int64_t n = 0; for (const PassBWindow& w : S->win) n += (int64_t)w.bonds.size(); return n; }
  if (!strncmp(key, "passb_lo", 8) && key[8] >= '0' && key[8] <= '7') { const size_t k = (size_t)(key[8] - '0'); return k < S->win.size() ? S->win[k].lo : -1; }
  if (!strncmp(key, "passb_mask", 10) && key[10] >= '0' && key[10] <= '7') { const size_t k = (size_t)(key[10] - '0'); return k < S->win.size() ? (int64_t)S->win[k].smask : -1; }
  if (!strncmp(key, "passb_nbonds", 12) && key[12] >= '0' && key[12] <= '7') { const size_t k = (size_t)(key[12] - '0'); return k < S->win.size() ? (int64_t)S->win[k].bonds.size() : -1; }
  if (!strncmp(key, "passb_items", 11) && key[11] >= '0' && key[11] <= '7') { const size_t k = (size_t)(key[11] - '0'); return k < S->win.size() ? (int64_t)S->win[k].nitems : -1; }
  if (!strcmp(key, "passb_ctas_used")) return S->win[0].ctas;
  if (!strcmp(key, "passb_lo")) return S->win[0].lo;
  if (!strcmp(key, "passb_s")) return S->win[0].s;
  if (!strcmp(key, "passb_items")) return S->win[0].nitems;
  if (!strcmp(key, "passb_smem")) return (int64_t)S->win[0].smem;
  return -1;
}

// Fill the host-side geometry of a window (classes, chunk sizes, item groups).  false if it cannot run
// (a popcount class does not fit shared memory even at X = 32, or the item count overflows 32 bits).
// Two CTAs per SM when every class fits half of the shared memory at X >= 32: one CTA's staging
// phase then overlaps the other's compute phase.
static bool passb_geometry(const ftlm_ctx* c, PassBWindow& w, std::vector<uint32_t>& grp_first) {
  const int N = c->N, K = c->N_up, esz = (int)ftlm_elem_size(c) * ftlm_plan_batch(c);   // bytes of one row of the batch
  w.f = N - w.lo - w.s;
  if (w.f < 0 || w.f > 20 || w.s < 2 || w.s > PASSB_MAX_S || w.lo < 0) return false;
  const int s1 = w.s + 1;
  w.ngroups = (1 << w.f) * s1;
  // largest class that actually occurs
  std::vector<char> used((size_t)s1, 0);
  for (uint32_t F = 0; F < (1u << w.f); ++F)
    for (int p = 0; p <= w.s; ++p) {
      const int kP = K - __builtin_popcount(F) - p;
      if (kP >= 0 && kP <= w.lo) used[(size_t)p] = 1;
    }
  w.max_conf = 0;
  for (int p = 0; p <= w.s; ++p) if (used[(size_t)p]) w.max_conf = std::max(w.max_conf, (int)binom_b(w.s, p));
  if (w.max_conf == 0) return false;
  const size_t fixed = passb_smem_bytes(N, K, w.max_conf, 0, esz);
  bool fits = false;
  int max_rows = 0;
  for (int ctas = c->passb_ctas > 0 ? c->passb_ctas : 2; ctas >= 1 && !fits; --ctas) {
    const size_t cap = (size_t)(228 * 1024) / (size_t)ctas - 1024 - (ctas == 1 ? 1024 : 0);
    if (fixed >= cap) continue;
    const size_t budget = cap - fixed;
    fits = true;
    max_rows = 0;
    for (int p = 0; p <= w.s && fits; ++p) {
      w.xk[p] = 0;
      if (!used[(size_t)p]) continue;
      const size_t per32 = (size_t)binom_b(w.s, p) * 32 * (size_t)esz;
      int xk = (int)std::min<size_t>(PASSB_XK, budget / per32);
      if (xk < 1) { fits = false; break; }
      w.xk[p] = xk;
      max_rows = std::max(max_rows, (int)binom_b(w.s, p) * 32 * xk);
    }
    if (fits) { w.ctas = ctas; w.threads = (ctas >= 2 || ftlm_elem_size(c) > 4) ? 512 : PASSB_THREADS; }
  }
  if (!fits) return false;
  w.smem = passb_smem_bytes(N, K, w.max_conf, max_rows, esz);
  grp_first.assign((size_t)w.ngroups + 1, 0);
  uint64_t total = 0;
  for (uint32_t F = 0; F < (1u << w.f); ++F)
    for (int p = 0; p <= w.s; ++p) {
      grp_first[(size_t)F * s1 + p] = (uint32_t)total;
      const int kP = K - __builtin_popcount(F) - p;
      if (kP < 0 || kP > w.lo) continue;
      const uint64_t RL = binom_b(w.lo, kP), X = 32ull * (uint64_t)w.xk[p];
      total += (RL + X - 1) / X;
      if (total >= 0xFFFFFFF0ull) return false;
    }
  grp_first[(size_t)w.ngroups] = (uint32_t)total;
  w.nitems = (uint32_t)total;
  return total > 0;
}

// Window selection = greedy cover of the candidate bonds (those with a site at or above mw, which the
// TML tile cannot serve from shared memory) by sets of at most smax label positions, all >= lo_min:
// grow a set from every uncovered bond by adding the position that brings in the most uncovered
// bonds (or, failing that, a neighbouring position), keep the best set, repeat while a window takes
// at least MIN_GAIN bonds (a window costs one more stream of v and y).
int ftlm_passb_plan_create(ftlm_ctx* c, int mw, const std::vector<int>& cand, std::vector<int>& window_of) {
  window_of.assign(cand.size(), -1);
  c->passb = nullptr;
  if (!c->use_passb || cand.empty()) return FTLM_OK;
  const int N = c->N;
  int smax = PASSB_MAX_S;                               // 12 for 4-byte rows; one position less per doubling of the row
  for (size_t rb = ftlm_elem_size(c) * (size_t)ftlm_plan_batch(c); rb > 4; rb >>= 1) --smax;
  if (c->passb_smax >= 2 && c->passb_smax < smax) smax = c->passb_smax;
  int lo_min = c->passb_lo_min > 0 ? c->passb_lo_min : std::max(8, mw - 7);
  if (lo_min > mw) lo_min = mw;
  const int MIN_GAIN = 3;
  PassBSet* S = new PassBSet();
  std::vector<std::vector<uint32_t>> groups;
  auto open_bond = [&](size_t k) {
    if (window_of[k] >= 0) return false;
    return c->bonds[(size_t)cand[k]].i >= lo_min;      // i < j
  };
  auto covered = [&](uint64_t set) {
    int n = 0;
    for (size_t k = 0; k < cand.size(); ++k)
      if (open_bond(k) && (c->bonds[(size_t)cand[k]].mask & ~set) == 0) ++n;
    return n;
  };
  for (;;) {
    uint64_t best_set = 0;
    int best_cnt = 0;
    auto grow = [&](uint64_t set) {
      int cur = covered(set);
      while (__builtin_popcountll(set) < smax) {
        int pick = -1, pick_cnt = cur;
        for (int v = lo_min; v < N; ++v) {
          if ((set >> v) & 1ull) continue;
          const int g = covered(set | (1ull << v));
          if (g > pick_cnt) { pick_cnt = g; pick = v; }
        }
        if (pick < 0) {                                   // no direct gain: a position next to the set
          for (size_t k = 0; k < cand.size() && pick < 0; ++k) {
            if (!open_bond(k)) continue;
            const uint64_t m = c->bonds[(size_t)cand[k]].mask;
            if ((m & set) != 0 && (m & ~set) != 0) pick = __builtin_ctzll(m & ~set);
          }
          if (pick < 0) break;
        }
        set |= 1ull << pick;
        cur = covered(set);
      }
      return set;
    };
    auto prune = [&](uint64_t set) {                      // keep only the positions some covered bond uses
      uint64_t used = 0;
      for (size_t k = 0; k < cand.size(); ++k)
        if (open_bond(k) && (c->bonds[(size_t)cand[k]].mask & ~set) == 0) used |= c->bonds[(size_t)cand[k]].mask;
      return used;
    };
    for (size_t seed = 0; seed < cand.size(); ++seed) {
      if (!open_bond(seed)) continue;
      uint64_t set = c->bonds[(size_t)cand[seed]].mask;
      for (int round = 0; round < 3; ++round) {           // positions that ended up unused are given back and re-spent
        const uint64_t before = set;
        set = prune(grow(set));
        if (set == before) break;
      }
      const int cur = covered(set);
      if (cur > best_cnt) { best_cnt = cur; best_set = set; }
    }
    if (best_cnt < MIN_GAIN) break;
    const uint64_t used = prune(best_set);
    PassBWindow w;
    w.smask = used;
    w.s = __builtin_popcountll(used);
    w.lo = __builtin_ctzll(used);                         // longest runs: every position below the window is passive
    if (N - w.lo - w.s > 20) break;
    std::vector<uint32_t> gf;
    if (!passb_geometry(c, w, gf)) break;
    const int widx = (int)S->win.size();
    for (size_t k = 0; k < cand.size() && (int)w.bonds.size() < PASSB_MAX_BONDS; ++k) {
      if (!open_bond(k)) continue;
      const BondDev& d = c->bonds[(size_t)cand[k]];
      if ((d.mask & ~w.smask) == 0) { window_of[k] = widx; w.bonds.push_back(cand[k]); w.Jh.push_back(d.Jh); }
    }
    S->win.push_back(w);
    groups.push_back(gf);
    if (S->win.size() >= 8) break;
  }
  if (S->win.empty()) { delete S; return FTLM_OK; }
  c->passb = S;
  // ---- tables + upload --------------------------------------------------------------------------
  for (size_t wi = 0; wi < S->win.size(); ++wi) {
    PassBWindow& w = S->win[wi];
    const int nU = 1 << w.s;
    std::vector<int> koff((size_t)w.s + 2, 0);
    for (int p = 0; p <= w.s; ++p) koff[(size_t)p + 1] = koff[(size_t)p] + (int)binom_b(w.s, p);
    std::vector<uint16_t> ustate((size_t)nU), slot((size_t)nU);
    std::vector<int> fill(koff.begin(), koff.end() - 1);
    for (int u = 0; u < nU; ++u) {                              // ascending u inside each popcount class
      const int p = __builtin_popcount((unsigned)u);
      slot[(size_t)u] = (uint16_t)(fill[(size_t)p] - koff[(size_t)p]);
      ustate[(size_t)fill[(size_t)p]++] = (uint16_t)u;
    }
    const size_t esz = ftlm_elem_size(c);
    std::vector<uint32_t> item_group((size_t)w.nitems);
    for (int g = 0; g < w.ngroups; ++g)
      for (uint32_t it = groups[wi][(size_t)g]; it < groups[wi][(size_t)g + 1]; ++it) item_group[it] = (uint32_t)g;
    std::vector<uint32_t> nbr((size_t)nU * 32, 0u);
    std::vector<double> nbrJ((size_t)nU * 32, 0.0);
    for (int u = 0; u < nU; ++u) {
      int n = 0;
      double sj = 0.0;
      const int pu = __builtin_popcount((unsigned)u);
      const int X = 32 * w.xk[pu];                                     // rows per tile row of this popcount class
      const size_t row = (size_t)koff[(size_t)pu] + slot[(size_t)u];    // position of u in window-word order (ustate)
      for (size_t e = 0; e < w.bonds.size(); ++e) {
        const BondDev& d = c->bonds[(size_t)w.bonds[e]];
        const uint32_t mk = (uint32_t)bits_extract(d.mask, w.smask), x = (uint32_t)u & mk;
        if (x != 0 && x != mk) {
          nbr[row * 32 + (size_t)n] = (uint32_t)slot[(size_t)((uint32_t)u ^ mk)] * (uint32_t)X;   // row index in the tile (the kernel scales by its row size)
          nbrJ[row * 32 + (size_t)n] = d.Jh;
          sj += d.Jh;
          ++n;
        }
      }
      // pad to a multiple of 4 with the word's own tile row: J = 0, or - uniform couplings, where the kernel adds first
      // and multiplies once - the common J with the added J * v[n] taken back through the sum of J
      const bool uni_w = [&] { for (size_t e = 1; e < w.Jh.size(); ++e) if (w.Jh[e] != w.Jh[0]) return false; return c->unij_allowed != 0 && !w.Jh.empty(); }();
      while (n & 3) {
        nbr[row * 32 + (size_t)n] = (uint32_t)slot[(size_t)u] * (uint32_t)X;
        nbrJ[row * 32 + (size_t)n] = 0.0;
        if (uni_w) sj += w.Jh[0];
        ++n;
      }
      nbr[row * 32 + 31] = (uint32_t)n;
      nbrJ[row * 32 + 31] = sj;
    }
    std::vector<float> nbrJf;
    if (esz == 4) { nbrJf.resize(nbrJ.size()); for (size_t k = 0; k < nbrJ.size(); ++k) nbrJf[k] = (float)nbrJ[k]; }
    auto up = [&](void** d, const void* h, size_t bytes) -> bool {
      if (ftlm_dmalloc(d, bytes ? bytes : 16) != cudaSuccess) return false;
      if (bytes && h && cudaMemcpy(*d, h, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return false;
      return true;
    };
    const size_t pbytes = (size_t)w.nitems * 24 * FTLM_MAX_BATCH;
    bool ok = up((void**)&w.d_ustate, ustate.data(), ustate.size() * 2) && up((void**)&w.d_koff, koff.data(), koff.size() * 4) &&
              up((void**)&w.d_nbr, nbr.data(), nbr.size() * 4) &&
              up(&w.d_nbrJ, esz == 4 ? (const void*)nbrJf.data() : (const void*)nbrJ.data(), nbrJ.size() * esz) &&
              up((void**)&w.d_grp_first, groups[wi].data(), groups[wi].size() * 4) &&
              up((void**)&w.d_item_group, item_group.data(), item_group.size() * 4) &&
              up((void**)&w.d_partials, nullptr, pbytes) && up((void**)&w.d_counter, nullptr, 16);
    if (ok) ok = cudaMemset(w.d_partials, 0, pbytes) == cudaSuccess && cudaMemset(w.d_counter, 0, 16) == cudaSuccess;
    if (!ok) { cudaGetLastError(); ftlm_passb_plan_destroy(c); ftlm_set_error("PASS-B: table upload failed"); return FTLM_ENOMEM; }
  }
  return FTLM_OK;
}

template <typename R, int B, int MODE>
static int launch_window(ftlm_ctx* c, PassBWindow& w, const void* v, void* y, int fused, cudaStream_t s) {
  PassBParams<R> p;
  memset(&p, 0, sizeof(p));
  p.N = c->N; p.K = c->N_up; p.lo = w.lo; p.s = w.s; p.f = w.f; p.ngroups = w.ngroups; p.nitems = w.nitems;
  p.dim = c->dim; p.binom = c->d_binom64; p.clt = c->d_clt; p.ustate = w.d_ustate; p.koff = w.d_koff;
  p.nbr_off = w.d_nbr; p.nbr_J = (const R*)w.d_nbrJ; p.grp_first = w.d_grp_first; p.item_group = w.d_item_group; p.partials = w.d_partials; p.counter = w.d_counter;
  p.st = c->d_state; p.max_conf = w.max_conf;
  p.unij = c->unij_allowed ? 1 : 0;
  for (size_t e = 1; e < w.Jh.size(); ++e) if (w.Jh[e] != w.Jh[0]) p.unij = 0;
  p.Juni = w.Jh.empty() ? (R)0 : (R)w.Jh[0];
  p.smask_hi = w.smask >> w.lo;
  p.fmask_hi = (c->N >= 64 ? ~0ull : ((1ull << c->N) - 1ull)) >> w.lo & ~p.smask_hi;
  for (int k = 0; k <= PASSB_MAX_S; ++k) p.xk[k] = w.xk[k];
  p.item_begin = 0; p.item_end = w.nitems;
  if (c->debug_item_count > 0) {
    p.item_begin = (uint32_t)std::min<int64_t>(c->debug_item_first, w.nitems);
    p.item_end = (uint32_t)std::min<int64_t>(c->debug_item_first + c->debug_item_count, w.nitems);
  }
  int grid = c->sm_count * w.ctas;
  if ((uint32_t)grid > p.item_end - p.item_begin) grid = (int)std::max(1u, p.item_end - p.item_begin);
  // 512 threads whenever the plan's rows are wider than 4 bytes (the launch bound of those kernels); a narrower run on
  // the same plan (remainder group, plan_batch) keeps that shape, so that the order of every sum is the same
  const int threads = (sizeof(R) * (size_t)ftlm_plan_batch(c) > 4) ? 512 : w.threads;
  if (fused) {
    auto k = passb_kernel<R, B, MODE, true>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)w.smem));
    FTLM_LAUNCH(k, grid, threads, w.smem, s, p, (const R*)v, (R*)y);
  } else {
    auto k = passb_kernel<R, B, MODE, false>;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)w.smem));
    FTLM_LAUNCH(k, grid, threads, w.smem, s, p, (const R*)v, (R*)y);
  }
  CK(cudaGetLastError());
  return FTLM_OK;
}

template <typename R, int B>
static int launch_window_m(ftlm_ctx* c, PassBWindow& w, const void* v, void* y, int fused, cudaStream_t s) {
  return c->mode == FTLM_INDEX_CLT ? launch_window<R, B, FTLM_INDEX_CLT>(c, w, v, y, fused, s)
                                   : launch_window<R, B, FTLM_INDEX_CR>(c, w, v, y, fused, s);
}

int ftlm_launch_passb(ftlm_ctx* c, const void* v, void* y, int fused, int batch, cudaStream_t s) {
  PassBSet* S = c->passb;
  if (!S) return FTLM_OK;
  if (batch > ftlm_plan_batch(c)) { ftlm_set_error("PASS-B: the window plan was built for %d chains, %d requested", ftlm_plan_batch(c), batch); return FTLM_EINVAL; }
  for (size_t wi = 0; wi < S->win.size(); ++wi) {
    PassBWindow& w = S->win[wi];
    if (!fused && c->debug_pass_mask && !((c->debug_pass_mask >> (wi + 1)) & 1)) continue;
    const int fz = (fused && wi + 1 == S->win.size()) ? 1 : 0;
    int rc;
    if (c->prec == FTLM_FP32) rc = batch == 1 ? launch_window_m<float, 1>(c, w, v, y, fz, s) : batch == 2 ? launch_window_m<float, 2>(c, w, v, y, fz, s) : launch_window_m<float, 4>(c, w, v, y, fz, s);
    else rc = batch == 1 ? launch_window_m<double, 1>(c, w, v, y, fz, s) : batch == 2 ? launch_window_m<double, 2>(c, w, v, y, fz, s) : launch_window_m<double, 4>(c, w, v, y, fz, s);
    if (rc != FTLM_OK) return rc;
  }
  return FTLM_OK;
}
