// Internal definitions shared by the CUDA translation units of libftlm (not part of the ABI).
#pragma once
#ifdef FTLM_EMU
// host SIMT emulation used by the -m "not gpu" tests (tests/emu/); never part of libftlm.so
#include "cuda_emu.h"
#else
#include <cuda_runtime.h>
#define FTLM_DYN_SMEM(name) extern __shared__ __align__(16) unsigned char name[]
#endif
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/ftlm.h"
#include "ftlm_access.cuh"

#ifndef FTLM_EMU
#ifdef FTLM_CHECKED
// checked build: every translation unit binds its copy of the check-state pointer before its first launch
FtlmChkState* ftlm_chk_state_dev();                 // device pointer of the process-wide state (ftlm_core.cu)
static inline void ftlm_chk_bind_tu() {
  static bool bound = false;
  if (!bound) { FtlmChkState* p = ftlm_chk_state_dev(); cudaMemcpyToSymbol(ftlm_chk_dev, &p, sizeof(p)); bound = true; }
}
#define FTLM_LAUNCH(kernel, grid, block, smem, stream, ...) (ftlm_chk_bind_tu(), kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__))
#else
#define FTLM_LAUNCH(kernel, grid, block, smem, stream, ...) kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__)
#endif
#endif

// Device allocations of the library go through these (the checked build keeps the table of live ranges
// that the kernels' address checks consult; otherwise they are cudaMalloc / cudaFree).
cudaError_t ftlm_dmalloc_bytes(void** p, size_t bytes);
template <typename T> static inline cudaError_t ftlm_dmalloc(T** p, size_t bytes) { return ftlm_dmalloc_bytes((void**)p, bytes); }
cudaError_t ftlm_dfree(void* p);
// Caller-owned device buffers an entry point is about to hand to kernels on stream `s` (checked build only).
void ftlm_chk_caller(cudaStream_t s, const void* p, size_t bytes);

#define FTLM_MAX_BONDS 4096
#define FTLM_MAX_BATCH 4

void ftlm_set_error(const char* fmt, ...);
int ftlm_cuda_fail(cudaError_t e, const char* what);

#define CK(call)                                                   \
  do {                                                             \
    cudaError_t e__ = (call);                                      \
    if (e__ != cudaSuccess) return ftlm_cuda_fail(e__, #call);     \
  } while (0)

// Device-resident scalars of one Lanczos chain (never read by the host between steps).
struct ChainState {
  double alpha[FTLM_MAX_STEPS];
  double beta[FTLM_MAX_STEPS];
  double scale;      // max_k(|alpha_k|, beta_k) so far (breakdown rule, reading 10)
  double beta_prev;  // beta_{j-1} used by the next fused H.v pass
  double a;          // alpha_j for the normalisation pass
  double inv_b;      // 1/beta_j for the normalisation pass
  double tol;
  double norm2;      // scratch: sum of squares (start-vector normalisation)
  int step;          // completed steps (= number of alphas stored)
  int limit;         // m = min(requested, dim)  (reading 9)
  int done;          // 1 after breakdown or once `limit` steps are done
  int pad;
};

struct BondDev {          // one bond as the kernels see it
  uint64_t mask;          // (1<<i) | (1<<j)
  double Jh;              // J_b / 2   (off-diagonal element on an antiparallel bond)
  double Jq;              // J_b / 4
  int i, j;               // i < j
};

// Three-level ("TML") kernel plans, built on the host in ftlm_create
// (DESIGN.md section 6).
struct TmlPlan;
struct PassBSet;
struct TmlrPlan;

struct ftlm_ctx {
  int N = 0, nb = 0, N_up = 0, mode = 0, prec = 0, device = 0;
  double h = 0.0;
  int64_t dim = 0;
  bool idx64 = false;     // indices need 64 bits (dim >= 2^32)
  bool lab64 = false;     // labels need 64 bits (N > 32)
  double diag0 = 0.0;     // sum_b J_b/4 - h*M_z : diagonal if every bond were parallel
  int sm_count = 148;

  // device tables
  uint64_t* d_binom64 = nullptr;   // [(N+1)][(N_up+1)] : C(p, a), exact
  uint32_t* d_binom32 = nullptr;   // same, saturated at 2^32-1 (used when !idx64)
  BondDev* d_bonds = nullptr;
  uint2* d_clt = nullptr;          // {M_b, C_b}
  int64_t n_clt = 0;
  uint64_t* d_lin_hi = nullptr;    // LIN mode: Ja[2^(N-h)] = number of sector labels with a smaller high half
  uint32_t* d_lin_lo = nullptr;    // LIN mode: Jb[2^h] = rank of the low half among the h-bit words of equal popcount
  int lin_h = 0;                   // low-half width N / 2
  std::vector<BondDev> bonds;
  std::vector<uint64_t> binom64;   // host copy

  // options
  int kernel = FTLM_KERNEL_AUTO;
  int tml_low_bits = 0, tml_mid_bits = 0;
  int use_persistent = 0;          // option "persistent": ftlm_lanczos runs small sectors with the one-launch chain kernel
  int use_graph = 0;               // option "graph": ftlm_chain_steps replays captured steps (CUDA graph)
  int graph_failed = 0;            // a capture / instantiate call failed on this handle: direct launches from then on
  int graph_roles[3] = {-1, -1, -1}, graph_batch = 0, graph_period = 0;   // what the cached graph was captured for
  void* graph_exec = nullptr;      // cudaGraphExec_t
  void* graph_stream = nullptr;    // capture stream (the caller's stream may be the legacy default stream)
  int graph_launches = 0;          // replays so far (read-only key "graph_launches")
  int allow_unverified = 0;        // option "allow_unverified": ftlm_autotune may run candidates without a device record
  uint64_t autotune_mask = 0;      // option "autotune_mask": bit k set = candidate k may run (0 = all); the ROW reference always runs
  int autotuned = 0;               // 1 + index of the candidate ftlm_autotune selected (0 = not tuned)
  double autotune_ms = 0.0;

  // three-level tile plan (ftlm_tml.cu)
  TmlPlan* tml = nullptr;
  // PASS-B windows for the bonds among the top label bits (ftlm_passb.cu); owned together with `tml`
  PassBSet* passb = nullptr;
  // in-tile pass with lane tables in registers (ftlm_tmlr.cu); exists only when every bond outside the
  // PASS-B windows stays inside the tile.  Option "tmlr": 1 = use it for the in-tile pass of kernel TML.
  TmlrPlan* tmlr = nullptr;
  int use_tmlr = 0;
  int unij_allowed = 1;            // option "tmlr_unij": 0 keeps the per-bond FMA form even on uniform-J lattices
  int use_passb = 0;               // option "passb": 1 moves the bonds that leave the tile into PASS-B windows (ftlm_autotune turns it on when it is valid and faster)
  int passb_lo_min = 0;            // option "passb_lo_min": lowest label position a window may use (0 = auto)
  int passb_smax = 0;              // option "passb_smax": largest window (0 = auto: 12 FP32 / 11 FP64)
  // test hooks (tests/emu runs sampled tiles / items of full-size sectors on the host): run only the
  // passes in the mask (bit 0 = TML pass, bit k+1 = PASS-B window k; 0 = all) and only the tiles /
  // items [first, first + count) (count 0 = all).  Non-fused H.v only.
  int debug_pass_mask = 0;
  int64_t debug_item_first = 0, debug_item_count = 0;
  int passb_ctas = 0;              // option "passb_ctas": CTAs per SM tried first (0 = auto: 2)

  // chain workspace
  void* q[3] = {nullptr, nullptr, nullptr};
  int ia = 0, ib = 1, ic = 2;      // q[ia] = q_j, q[ib] = q_{j-1}, q[ic] = y
  bool pending_norm = false;       // lazy normalisation: q_{j+1} = (q[ic] - alpha_j q[ia]) / beta_j is not materialised yet
  int lazy_norm = 0;               // option "lazy_norm": 1 = the TMLR pass forms q_{j+1} while staging (no normalisation pass)
  ChainState* d_state = nullptr;   // [FTLM_MAX_BATCH]
  double* d_partials = nullptr;    // [3 * FTLM_MAX_BATCH][max_blocks]
  unsigned int* d_ticket = nullptr;  // [FTLM_MAX_BATCH]
  int batch = 1;                   // option "batch": chains ftlm_lanczos advances together on interleaved vectors (1, 2, 4)
  int plan_batch = 0;              // option "plan_batch": build the tile / window plans for this many chains even when fewer run (0 = follow "batch")
  int cur_batch = 1;               // batch of the chain(s) in progress
  int q_batch = 0;                 // batch the work vectors were allocated for
  int max_blocks = 0;
  int steps_enqueued = 0;
  int chain_limit = 0;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
};

size_t ftlm_elem_size(const ftlm_ctx* c);
int ftlm_effective_kernel(const ftlm_ctx* c);

// ---- launches implemented in the kernel translation units -------------------------------
// fused == 0: y = H v.   fused == 1: y = H q - beta_prev q_prev with the three FP64 sums and
// the in-kernel finalisation of alpha_j, beta_j into ctx->d_state.
int ftlm_launch_hv_row(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, int batch, cudaStream_t s);
int ftlm_launch_neighbors_row(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s);
// ROWG: unrank once per 8 consecutive rows, Gosper-style successor in between (single vector)
int ftlm_launch_hv_rowg(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, cudaStream_t s);
int ftlm_launch_neighbors_rowg(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s);

int ftlm_tml_plan_create(ftlm_ctx* c);
void ftlm_tml_plan_destroy(ftlm_ctx* c);
int64_t ftlm_tml_info(const ftlm_ctx* c, const char* key);
int ftlm_launch_hv_tml(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, int batch, cudaStream_t s);
int ftlm_launch_neighbors_tml(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, cudaStream_t s);

int ftlm_tmlr_plan_create(ftlm_ctx* c, int w, int m, const std::vector<int>& in_window);
void ftlm_tmlr_plan_destroy(ftlm_ctx* c);
int64_t ftlm_tmlr_info(const ftlm_ctx* c, const char* key);
int ftlm_launch_hv_tmlr(ftlm_ctx* c, const void* v, const void* qprev, void* y, int fused, cudaStream_t s);
// Lazy-normalisation form of the fused pass: yq holds y_j on entry and q_{j+1} = (y_j - alpha_j q_j)/beta_j on
// exit (formed while the tile is staged); q = q_j (also the q_prev of this step); y receives the pass's output.
int ftlm_launch_hv_tmlr_lazy(ftlm_ctx* c, void* yq, const void* q, void* y, int fused, cudaStream_t s);
bool ftlm_tmlr_lazy_ok(const ftlm_ctx* c);

// Persistent chain kernel (ftlm_chain.cu): whole Lanczos chains of a small sector in one launch, one CTA per chain,
// the three work vectors in shared memory.  ftlm_chain_persistent_fits: the sector fits; the launch runs chains
// r0 .. r0 + nchains - 1 for `limit` steps and leaves alpha / beta / step counts in d_alpha, d_beta [nchains][limit], d_m_eff.
bool ftlm_chain_persistent_fits(const ftlm_ctx* c);
int ftlm_launch_chain_persistent(ftlm_ctx* c, uint64_t seed, int r0, int nchains, int limit, double* d_alpha, double* d_beta,
                                 int* d_m_eff, cudaStream_t s);

// PASS-B (ftlm_passb.cu).  `tt` lists the bonds whose two sites lie at positions >= mw (candidate
// top-top bonds) as indices into c->bonds; on return window_of[k] is the PASS-B window that took
// tt[k] or -1 if the bond stays in the TML kernel.  FTLM_OK with c->passb == nullptr if no window pays.
int ftlm_passb_plan_create(ftlm_ctx* c, int mw, const std::vector<int>& tt, std::vector<int>& window_of);
void ftlm_passb_plan_destroy(ftlm_ctx* c);
int ftlm_passb_windows(const ftlm_ctx* c);
void ftlm_passb_window_geometry(const ftlm_ctx* c, int window, int* lo, int* s);
int64_t ftlm_passb_info(const ftlm_ctx* c, const char* key);
// y += sum over the windows' bonds of (J_b/2)(P_b - 1) v.  fused: the last window also accumulates the
// three FP64 sums over the final y and advances the chain state.
int ftlm_launch_passb(ftlm_ctx* c, const void* v, void* y, int fused, int batch, cudaStream_t s);
// chains the plans (tile split, window sizes) are built for
static inline int ftlm_plan_batch(const ftlm_ctx* c) { return c->plan_batch > c->batch ? c->plan_batch : c->batch; }

// ---- device helpers ---------------------------------------------------------------------
#ifdef __CUDACC__

// counter-based start-vector generator: element t of the chain with key `key`
#define FTLM_GOLD 0x9E3779B97F4A7C15ull
__device__ __forceinline__ uint64_t mix64(uint64_t x) {
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}
__device__ __forceinline__ double gauss_elem(uint64_t key, uint64_t t) {
  const uint64_t a = mix64(key + FTLM_GOLD * (2ull * t + 1ull));
  const uint64_t b = mix64(key + FTLM_GOLD * (2ull * t + 2ull));
  const double u1 = ((double)(a >> 11) + 1.0) * 0x1.0p-53;
  const double u2 = (double)(b >> 11) * 0x1.0p-53;
  return sqrt(-2.0 * log(u1)) * cos(6.283185307179586 * u2);
}

__device__ __forceinline__ int popc_(uint32_t x) { return __popc(x); }
__device__ __forceinline__ int popc_(uint64_t x) { return __popcll(x); }
__device__ __forceinline__ int ffs_(uint32_t x) { return __ffs((int)x); }
__device__ __forceinline__ int ffs_(uint64_t x) { return __ffsll((long long)x); }

// asynchronous global -> shared copy of one element (LDGSTS); the emulation copies at once
template <typename T>
__device__ __forceinline__ void cp_async_elem_(T* smem_dst, const T* gsrc, int line) {
  if (!FTLM_SW_OK(smem_dst, T, line) || !FTLM_G_OK(gsrc, T, line)) return;
#ifdef FTLM_EMU
  cuda_emu::cp_async_issue(smem_dst, gsrc, sizeof(T));
#else
  static_assert(sizeof(T) == 4 || sizeof(T) == 8 || sizeof(T) == 16, "cp.async copies 4, 8 or 16 bytes");
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (sizeof(T) == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(gsrc) : "memory");
  else if (sizeof(T) == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
  else asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
#endif
}
#define cp_async_elem(dst, src) cp_async_elem_((dst), (src), __LINE__)
__device__ __forceinline__ void cp_async_wait_all() {
#ifdef FTLM_EMU
  cuda_emu::cp_async_wait_all();      // the copies of the calling thread land here, not before
#else
  asm volatile("cp.async.wait_all;" ::: "memory");
#endif
}

// ---- bulk copy global -> shared with mbarrier completion (Blackwell/Hopper async proxy; SASS UBLKCP + SYNCS) -----
// One thread announces the bytes (arrive.expect_tx) and issues the copy; every thread of the CTA waits on the phase
// parity.  Source, destination and size are multiples of 16 bytes.  The emulation lands the bytes at the first wait
// that finds the phase complete (destination poisoned until then).
__device__ __forceinline__ void mbar_init(uint64_t* mbar, int count) {
#ifdef FTLM_EMU
  cuda_emu::mbar_init(mbar, count);
#else
  const unsigned a = (unsigned)__cvta_generic_to_shared(mbar);
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#endif
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* mbar, uint32_t bytes) {
#ifdef FTLM_EMU
  cuda_emu::mbar_arrive_expect_tx(mbar, bytes);
#else
  const unsigned a = (unsigned)__cvta_generic_to_shared(mbar);
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
#endif
}
__device__ __forceinline__ void bulk_copy_g2s_(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* mbar, int line) {
  if (!FTLM_S_OKN(smem_dst, bytes, 16, line) || !FTLM_G_OKN(gsrc, bytes, 16, line)) {
    // checked build: the copy is suppressed; its bytes are taken back from the barrier so that nobody waits for them
#if defined(FTLM_CHECKED) && !defined(FTLM_EMU)
    const unsigned a = (unsigned)__cvta_generic_to_shared(mbar);
    asm volatile("mbarrier.complete_tx.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
#endif
    return;
  }
#ifdef FTLM_EMU
  cuda_emu::bulk_issue(smem_dst, gsrc, bytes, mbar, FTLM_TU, line);
#else
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst), a = (unsigned)__cvta_generic_to_shared(mbar);
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(d), "l"(gsrc), "r"(bytes), "r"(a) : "memory");
#endif
}
#define bulk_copy_g2s(dst, src, bytes, mbar) bulk_copy_g2s_((dst), (src), (bytes), (mbar), __LINE__)
__device__ __forceinline__ void mbar_wait(uint64_t* mbar, uint32_t parity) {
#ifdef FTLM_EMU
  cuda_emu::mbar_wait(mbar, parity);
#else
  const unsigned a = (unsigned)__cvta_generic_to_shared(mbar);
  unsigned done = 0;
  while (!done) {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(a), "r"(parity) : "memory");
  }
#endif
}

__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
  return x;
}

// Deterministic block sum of three doubles (fixed tree). Result valid in thread 0.
// `sh` must hold 3*32 doubles.
__device__ __forceinline__ void block_sum3(double& a, double& b, double& c, double* sh) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
  __syncthreads();
  if (lane == 0) { sh[w] = a; sh[32 + w] = b; sh[64 + w] = c; }
  __syncthreads();
  if (w == 0) {
    a = lane < nw ? sh[lane] : 0.0;
    b = lane < nw ? sh[32 + lane] : 0.0;
    c = lane < nw ? sh[64 + lane] : 0.0;
    a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
  }
}

// Grid-wide deterministic finish of the fused Lanczos reductions (H9): every block stores its
// three partial sums, the last block to arrive (ticket) adds them in block order with a fixed
// tree and advances the chain state: alpha_j = <q,y>/<q,q>, beta_j^2 = <y,y> - <q,y>^2/<q,q>
// (H5(i): never assumes ||q|| = 1), breakdown rule of reading 10.
__device__ __forceinline__ void lanczos_finish(double s_qy, double s_yy, double s_qq, double* partials,
                                               int stride, unsigned int* ticket, ChainState* st,
                                               double* sh) {
  block_sum3(s_qy, s_yy, s_qq, sh);
  __shared__ bool last;
  if (threadIdx.x == 0) {
    ST_G(&partials[blockIdx.x], s_qy);
    ST_G(&partials[stride + blockIdx.x], s_yy);
    ST_G(&partials[2 * stride + blockIdx.x], s_qq);
    __threadfence();
    last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double a = 0.0, b = 0.0, c = 0.0;
  for (int k = threadIdx.x; k < (int)gridDim.x; k += blockDim.x) {   // fixed assignment + order
    a += LD_G(&partials[k]); b += LD_G(&partials[stride + k]); c += LD_G(&partials[2 * stride + k]);
  }
  block_sum3(a, b, c, sh);
  if (threadIdx.x == 0) {
    *ticket = 0;
    if (st->done) return;                 // a chain of a batch that broke down earlier keeps its coefficients
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

#endif  // __CUDACC__
