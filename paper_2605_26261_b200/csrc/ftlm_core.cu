// libftlm core: handle, sector tables (A0/A1), start vectors, the fused Lanczos chain driver
// and the C-ABI entry points that dispatch to the ROW / TML kernels.
#include <algorithm>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstring>

#define FTLM_TU 1
#include "ftlm_common.cuh"

static void graph_drop(ftlm_ctx* c);                 // cached CUDA graph of the chain step (defined with ftlm_chain_steps)

// ---- errors --------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

void ftlm_set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
int ftlm_cuda_fail(cudaError_t e, const char* what) {
  ftlm_set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
  return FTLM_ECUDA;
}
extern "C" const char* ftlm_last_error(void) { return g_err; }
#ifdef FTLM_CHECKED
extern "C" const char* ftlm_version(void) { return "ftlm-b200 0.3 (sm_100a) CHECKED"; }
#else
extern "C" const char* ftlm_version(void) { return "ftlm-b200 0.3 (sm_100a)"; }
#endif

// ---- device allocations; checked build: table of live ranges (ftlm_access.cuh) -------------------
#if defined(FTLM_CHECKED) && !defined(FTLM_EMU)
#include <algorithm>
#include <mutex>
namespace {
std::mutex g_chk_mu;
FtlmChkState* g_chk_dev = nullptr;
std::vector<FtlmChkRange> g_chk_lib;                 // sorted by lo
FtlmChkRange g_chk_call[FTLM_CHK_CALL_RANGES];
int g_chk_call_next = 0;

void chk_upload_lib() {                              // allocation / free: no kernel of this library may be in flight on a freed range anyway
  struct { int n, pad; } head = {(int)g_chk_lib.size(), 0};
  cudaDeviceSynchronize();
  cudaMemcpy((char*)g_chk_dev + offsetof(FtlmChkState, ranges), g_chk_lib.data(), sizeof(FtlmChkRange) * g_chk_lib.size(), cudaMemcpyHostToDevice);
  cudaMemcpy((char*)g_chk_dev + offsetof(FtlmChkState, n_ranges), &head, sizeof(head), cudaMemcpyHostToDevice);
}
}  // namespace

FtlmChkState* ftlm_chk_state_dev() {
  std::lock_guard<std::mutex> lk(g_chk_mu);
  if (!g_chk_dev) {
    if (cudaMalloc((void**)&g_chk_dev, sizeof(FtlmChkState)) != cudaSuccess) { g_chk_dev = nullptr; return nullptr; }
    cudaMemset(g_chk_dev, 0, sizeof(FtlmChkState));
    memset(g_chk_call, 0, sizeof(g_chk_call));
  }
  return g_chk_dev;
}

cudaError_t ftlm_dmalloc_bytes(void** p, size_t bytes) {
  cudaError_t e = cudaMalloc(p, bytes);
  if (e != cudaSuccess) return e;
  if (!ftlm_chk_state_dev()) return cudaErrorMemoryAllocation;
  std::lock_guard<std::mutex> lk(g_chk_mu);
  if (g_chk_lib.size() >= FTLM_CHK_MAX_RANGES) { cudaFree(*p); *p = nullptr; return cudaErrorMemoryAllocation; }
  const FtlmChkRange r{(unsigned long long)*p, (unsigned long long)*p + bytes};
  g_chk_lib.insert(std::upper_bound(g_chk_lib.begin(), g_chk_lib.end(), r, [](const FtlmChkRange& a, const FtlmChkRange& b) { return a.lo < b.lo; }), r);
  chk_upload_lib();
  return cudaSuccess;
}

cudaError_t ftlm_dfree(void* p) {
  if (p) {
    std::lock_guard<std::mutex> lk(g_chk_mu);
    for (size_t k = 0; k < g_chk_lib.size(); ++k)
      if (g_chk_lib[k].lo == (unsigned long long)p) { g_chk_lib.erase(g_chk_lib.begin() + (long)k); break; }
    if (g_chk_dev) chk_upload_lib();
  }
  return cudaFree(p);
}

void ftlm_chk_caller(cudaStream_t s, const void* p, size_t bytes) {
  if (!p || !bytes || !ftlm_chk_state_dev()) return;
  std::lock_guard<std::mutex> lk(g_chk_mu);
  const FtlmChkRange r{(unsigned long long)p, (unsigned long long)p + bytes};
  for (int k = 0; k < FTLM_CHK_CALL_RANGES; ++k)
    if (g_chk_call[k].lo == r.lo && g_chk_call[k].hi == r.hi) return;   // already listed
  g_chk_call[g_chk_call_next] = r;
  g_chk_call_next = (g_chk_call_next + 1) % FTLM_CHK_CALL_RANGES;
  // stream-ordered: kernels already enqueued keep the list they were launched under (pageable source: staged at once)
  cudaMemcpyAsync((char*)g_chk_dev + offsetof(FtlmChkState, call), g_chk_call, sizeof(g_chk_call), cudaMemcpyHostToDevice, s);
}

// Self-test of the checker ("check_selftest"): five accesses that would fault in the release build - a global load and a
// global store outside every live range, a misaligned global load, a shared load beyond the dynamic window, an
// asynchronous copy from a bad source - must each be suppressed and counted.  Returns how many were counted (5)
// and puts the counter back, so that a session's "violations == 0" criterion is not disturbed.
__global__ void chk_selftest_kernel(const float* good, float* sink) {
  FTLM_DYN_SMEM(smem);
  float* sm = (float*)smem;
  if (threadIdx.x == 0) {
    float a = LD_G(good + (1ll << 40));                       // far outside
    ST_G((float*)(uintptr_t)64, 1.0f);                         // unmapped low address
    a += LD_G((const float*)((const char*)good + 2));         // misaligned
    a += LD_S(sm + (1 << 20));                                 // beyond the dynamic shared-memory window
    cp_async_elem(sm, (const float*)(uintptr_t)128);
    cp_async_wait_all();
    ST_G(sink, a + LD_G(good));                                // legitimate accesses: not counted
  }
}

static int64_t chk_selftest() {
  if (!ftlm_chk_state_dev()) return -1;
  float* buf = nullptr;
  if (ftlm_dmalloc(&buf, 64) != cudaSuccess) return -1;
  cudaMemset(buf, 0, 64);
  unsigned long long before = 0, after = 0;
  cudaDeviceSynchronize();
  cudaMemcpy(&before, g_chk_dev, 8, cudaMemcpyDeviceToHost);
  FTLM_LAUNCH(chk_selftest_kernel, 1, 32, 64, 0, buf, buf + 8);
  const cudaError_t e = cudaDeviceSynchronize();
  cudaMemcpy(&after, g_chk_dev, 8, cudaMemcpyDeviceToHost);
  FtlmChkState zero;
  memset(&zero, 0, sizeof(zero));
  if (before == 0) cudaMemcpy(g_chk_dev, &zero, offsetof(FtlmChkState, n_ranges), cudaMemcpyHostToDevice);   // forget the deliberate ones
  else cudaMemcpy(g_chk_dev, &before, 8, cudaMemcpyHostToDevice);
  ftlm_dfree(buf);
  return e == cudaSuccess ? (int64_t)(after - before) : -2;
}

static int64_t chk_read(const char* key) {
  if (!ftlm_chk_state_dev()) return -1;
  if (!strcmp(key, "check_selftest")) return chk_selftest();
  FtlmChkState h;
  cudaDeviceSynchronize();
  if (cudaMemcpy(&h, g_chk_dev, offsetof(FtlmChkState, call), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
  if (!strcmp(key, "check_violations")) return (int64_t)h.violations;
  if (!strcmp(key, "check_first_tu")) return h.first_tu;
  if (!strcmp(key, "check_first_line")) return h.first_line;
  if (!strcmp(key, "check_first_kind")) return h.first_kind;
  if (!strcmp(key, "check_first_block")) return h.first_block;
  if (!strcmp(key, "check_first_thread")) return h.first_thread;
  if (!strcmp(key, "check_first_addr")) return (int64_t)h.first_addr;
  return -1;
}
#else
cudaError_t ftlm_dmalloc_bytes(void** p, size_t bytes) { return cudaMalloc(p, bytes); }
cudaError_t ftlm_dfree(void* p) { return cudaFree(p); }
void ftlm_chk_caller(cudaStream_t, const void*, size_t) {}
#endif

size_t ftlm_elem_size(const ftlm_ctx* c) { return c->prec == FTLM_FP64 ? 8 : 4; }

// ---- CLT construction (A1; L150-L154, Eq. 18) --------------------------------------------
// For d = 2 the occupancy mask of block b depends only on N_up - popc(b) and C_b is the number
// of sector labels below 32 b, so every block is built independently (no scan):
//   M_b bit j = [popc(j) == N_up - popc(b)],  C_b = sum over set bits p of 32b (from the top) of
//   C(p, N_up - ones_above).  Equals the paper's "set bits, then cumulative sum" construction.
__global__ void clt_build_kernel(uint2* __restrict__ clt, int64_t nblk, int N, int K,
                                 const uint64_t* __restrict__ binom) {
  const int K1 = K + 1;
  for (int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; b < nblk;
       b += (int64_t)gridDim.x * blockDim.x) {
    const int want = K - __popcll((unsigned long long)b);
    uint32_t mask = 0;
    if (want >= 0 && want <= 5) {
      for (int j = 0; j < 32; ++j)
        if (__popc(j) == want && (N >= 5 || j < (1 << N))) mask |= 1u << j;
    }
    const uint64_t base = (uint64_t)b << 5;
    uint64_t cnt = 0;
    int above = 0;
    for (int p = N - 1; p >= 5; --p) {
      if ((base >> p) & 1ull) {
        const int need = K - above;
        if (need >= 0 && need <= p) cnt += LDG(&binom[p * K1 + need]);
        ++above;
      }
    }
    ST_G(&clt[b], make_uint2(mask, (uint32_t)cnt));
  }
}

// ---- start vectors (readings 12-14) ---------------------------------------
static uint64_t mix64_host(uint64_t x) {
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}

__global__ void __launch_bounds__(256)
gauss_norm_kernel(uint64_t key, int64_t dim, double* __restrict__ partials) {
  __shared__ double sh[96];
  double s = 0.0, z1 = 0.0, z2 = 0.0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < dim;
       t += (int64_t)gridDim.x * blockDim.x) {
    const double g = gauss_elem(key, (uint64_t)t);
    s += g * g;
  }
  block_sum3(s, z1, z2, sh);
  if (threadIdx.x == 0) ST_G(&partials[blockIdx.x], s);
}

template <typename R>
__global__ void __launch_bounds__(256)
sumsq_kernel(const R* __restrict__ v, int64_t dim, double* __restrict__ partials) {
  __shared__ double sh[96];
  double s = 0.0, z1 = 0.0, z2 = 0.0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < dim;
       t += (int64_t)gridDim.x * blockDim.x) {
    const double g = (double)LD_G(&v[t]);
    s += g * g;
  }
  block_sum3(s, z1, z2, sh);
  if (threadIdx.x == 0) ST_G(&partials[blockIdx.x], s);
}

__global__ void reduce_partials_kernel(const double* __restrict__ partials, int n, double* out) {
  __shared__ double sh[96];
  double s = 0.0, z1 = 0.0, z2 = 0.0;
  for (int k = threadIdx.x; k < n; k += blockDim.x) s += LD_G(&partials[k]);
  block_sum3(s, z1, z2, sh);
  if (threadIdx.x == 0) *out = s;
}

template <typename R>
__global__ void __launch_bounds__(256)
gauss_write_kernel(uint64_t key, int64_t dim, const double* __restrict__ norm2, R* __restrict__ v, int vstride, int voff) {
  const double nrm = sqrt(*norm2);                       // element t of the chain goes to v[t * vstride + voff] (interleaved batch)
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < dim;
       t += (int64_t)gridDim.x * blockDim.x)
    ST_G(&v[t * vstride + voff], (R)(gauss_elem(key, (uint64_t)t) / nrm));
}

template <typename R>
__global__ void __launch_bounds__(256)
scale_copy_kernel(const R* __restrict__ src, int64_t dim, const double* __restrict__ norm2, R* __restrict__ dst, int dstride, int doff) {
  const double nrm = sqrt(*norm2);
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < dim;
       t += (int64_t)gridDim.x * blockDim.x)
    ST_G(&dst[t * dstride + doff], (R)((double)LD_G(&src[t]) / nrm));
}

// ---- Lanczos normalisation pass (A7): q_{j+1} = (y - alpha_j q_j) / beta_j ----------------------
// B interleaved chains: element i of the arrays belongs to chain i % B and uses that chain's alpha_j, 1 / beta_j
// (a chain that has broken down has 1 / beta = 0: its column becomes zero and stays out of the way).
template <typename R, typename V4, int B>
__global__ void __launch_bounds__(256)
lanczos_next_kernel(const R* __restrict__ y, const R* __restrict__ q, R* __restrict__ qnext,
                    int64_t dim, const ChainState* __restrict__ st) {
  bool all_done = true;
  R av[B], ibv[B];
#pragma unroll
  for (int c = 0; c < B; ++c) { all_done = all_done && st[c].done; av[c] = (R)st[c].a; ibv[c] = (R)st[c].inv_b; }
  if (all_done) return;
  constexpr int W = sizeof(V4) / sizeof(R);
  const int64_t nvec = dim / W;
  const V4* y4 = (const V4*)y;
  const V4* q4 = (const V4*)q;
  V4* o4 = (V4*)qnext;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < nvec; k += stride) {
    V4 yy = LDCS(&y4[k]);
    V4 qq = LD_G(&q4[k]);
    R* yp = (R*)&yy;
    const R* qp = (const R*)&qq;
#pragma unroll
    for (int e = 0; e < W; ++e) {
      const int c = B == 1 ? 0 : (int)((k * W + e) % B);
      R a = av[0], ib = ibv[0];
#pragma unroll
      for (int cc = 1; cc < B; ++cc) if (c == cc) { a = av[cc]; ib = ibv[cc]; }
      yp[e] = (yp[e] - a * qp[e]) * ib;
    }
    ST_G(&o4[k], yy);
  }
  for (int64_t t = nvec * W + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < dim; t += stride) {
    const int c = B == 1 ? 0 : (int)(t % B);
    R a = av[0], ib = ibv[0];
#pragma unroll
    for (int cc = 1; cc < B; ++cc) if (c == cc) { a = av[cc]; ib = ibv[cc]; }
    ST_G(&qnext[t], (LD_G(&y[t]) - a * LD_G(&q[t])) * ib);
  }
}

__global__ void chain_reset_kernel(ChainState* st0, int limit, double tol, int nb) {
  if (blockIdx.x == 0 && (int)threadIdx.x < nb) {
    ChainState* st = st0 + threadIdx.x;
    st->scale = 0.0; st->beta_prev = 0.0; st->a = 0.0; st->inv_b = 0.0; st->tol = tol;
    st->step = 0; st->limit = limit; st->done = (limit <= 0);
  }
}

// ---- handle ------------------------------------------------------------------------------------
static uint64_t binom_u64(int n, int k) {
  if (k < 0 || k > n) return 0;
  if (k > n - k) k = n - k;
  unsigned __int128 r = 1;
  for (int i = 1; i <= k; ++i) r = r * (unsigned)(n - k + i) / (unsigned)i;
  return (uint64_t)r;
}

extern "C" int ftlm_create(ftlm_ctx** out, int N, int n_bonds, const int32_t* bond_i, const int32_t* bond_j,
                           const double* J, double h, int N_up, int index_mode, int precision, int device) {
  if (!out) { ftlm_set_error("ftlm_create: out is NULL"); return FTLM_EINVAL; }
  *out = nullptr;
  if (N < 1 || N > 62) { ftlm_set_error("ftlm_create: N=%d outside [1,62]", N); return FTLM_EINVAL; }
  if (N_up < 0 || N_up > N) { ftlm_set_error("ftlm_create: N_up=%d outside [0,%d]", N_up, N); return FTLM_EINVAL; }
  if (n_bonds < 0 || n_bonds > FTLM_MAX_BONDS || (n_bonds > 0 && (!bond_i || !bond_j || !J))) {
    ftlm_set_error("ftlm_create: bad bond list (n_bonds=%d)", n_bonds); return FTLM_EINVAL;
  }
  if (index_mode != FTLM_INDEX_CLT && index_mode != FTLM_INDEX_CR && index_mode != FTLM_INDEX_LIN) { ftlm_set_error("ftlm_create: bad index_mode %d", index_mode); return FTLM_EINVAL; }
  if (precision != FTLM_FP32 && precision != FTLM_FP64) { ftlm_set_error("ftlm_create: bad precision %d", precision); return FTLM_EINVAL; }
  for (int b = 0; b < n_bonds; ++b) {
    if (bond_i[b] < 0 || bond_i[b] >= N || bond_j[b] < 0 || bond_j[b] >= N || bond_i[b] == bond_j[b]) {
      ftlm_set_error("ftlm_create: bond %d = (%d,%d) invalid for N=%d", b, bond_i[b], bond_j[b], N);
      return FTLM_EINVAL;
    }
  }
  if (index_mode == FTLM_INDEX_CLT && N > 32) { ftlm_set_error("ftlm_create: CLT needs N <= 32 (got %d); use CR", N); return FTLM_EUNSUPPORTED; }
  if (index_mode == FTLM_INDEX_LIN && N > 48) { ftlm_set_error("ftlm_create: LIN needs N <= 48 (got %d); use CR", N); return FTLM_EUNSUPPORTED; }
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev <= 0) {
    ftlm_set_error("ftlm_create: no CUDA device (%s); this library has no CPU path", cudaGetErrorString(e));
    return FTLM_ECUDA;
  }
  if (device < 0 || device >= ndev) { ftlm_set_error("ftlm_create: device %d of %d", device, ndev); return FTLM_EINVAL; }
  CK(cudaSetDevice(device));

  ftlm_ctx* c = new ftlm_ctx();
  c->N = N; c->nb = n_bonds; c->N_up = N_up; c->mode = index_mode; c->prec = precision; c->device = device; c->h = h;
  c->dim = (int64_t)binom_u64(N, N_up);
  c->idx64 = (uint64_t)c->dim >= (1ull << 32);
  c->lab64 = N > 32;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) c->sm_count = prop.multiProcessorCount;

  double sumJq = 0.0;
  c->bonds.resize(n_bonds);
  for (int b = 0; b < n_bonds; ++b) {
    BondDev& d = c->bonds[b];
    d.i = bond_i[b] < bond_j[b] ? bond_i[b] : bond_j[b];
    d.j = bond_i[b] < bond_j[b] ? bond_j[b] : bond_i[b];
    d.mask = (1ull << d.i) | (1ull << d.j);
    d.Jh = 0.5 * J[b]; d.Jq = 0.25 * J[b];
    sumJq += d.Jq;
  }
  c->diag0 = sumJq - h * ((double)N_up - 0.5 * (double)N);

  const int K1 = N_up + 1;
  c->binom64.assign((size_t)(N + 1) * K1, 0);
  std::vector<uint32_t> b32((size_t)(N + 1) * K1, 0);
  for (int p = 0; p <= N; ++p)
    for (int a = 0; a <= N_up; ++a) {
      const uint64_t v = binom_u64(p, a);
      c->binom64[(size_t)p * K1 + a] = v;
      b32[(size_t)p * K1 + a] = v > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)v;
    }
  int rc = FTLM_OK;
  auto fail = [&](int code) { ftlm_destroy(c); return code; };
#define CKF(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = ftlm_cuda_fail(e__, #call); return fail(e__ == cudaErrorMemoryAllocation ? FTLM_ENOMEM : rc); } } while (0)
  CKF(ftlm_dmalloc(&c->d_binom64, c->binom64.size() * 8));
  CKF(ftlm_dmalloc(&c->d_binom32, b32.size() * 4));
  CKF(cudaMemcpy(c->d_binom64, c->binom64.data(), c->binom64.size() * 8, cudaMemcpyHostToDevice));
  CKF(cudaMemcpy(c->d_binom32, b32.data(), b32.size() * 4, cudaMemcpyHostToDevice));
  CKF(ftlm_dmalloc(&c->d_bonds, sizeof(BondDev) * (size_t)(n_bonds > 0 ? n_bonds : 1)));
  if (n_bonds > 0) CKF(cudaMemcpy(c->d_bonds, c->bonds.data(), sizeof(BondDev) * n_bonds, cudaMemcpyHostToDevice));
  c->max_blocks = c->sm_count * 32;
  CKF(ftlm_dmalloc(&c->d_state, sizeof(ChainState) * FTLM_MAX_BATCH));
  CKF(cudaMemset(c->d_state, 0, sizeof(ChainState) * FTLM_MAX_BATCH));
  CKF(ftlm_dmalloc(&c->d_partials, sizeof(double) * 3 * FTLM_MAX_BATCH * (size_t)c->max_blocks));
  CKF(ftlm_dmalloc(&c->d_ticket, sizeof(unsigned int) * FTLM_MAX_BATCH));
  CKF(cudaMemset(c->d_ticket, 0, sizeof(unsigned int) * FTLM_MAX_BATCH));
  if (index_mode == FTLM_INDEX_CLT) {
    c->n_clt = (int64_t)(((1ull << N) + 31ull) / 32ull);
    CKF(ftlm_dmalloc(&c->d_clt, sizeof(uint2) * (size_t)c->n_clt));
    int grid = (int)((c->n_clt + 255) / 256);
    if (grid > c->sm_count * 16) grid = c->sm_count * 16;
    FTLM_LAUNCH(clt_build_kernel, grid, 256, 0, 0, c->d_clt, c->n_clt, N, N_up, c->d_binom64);
    CKF(cudaGetLastError());
  }
  if (index_mode == FTLM_INDEX_LIN) {
    // Lin's two tables (L119) in the ascending-label order: Ja by a running count over the high halves
    // (C(h, N_up - popc(a)) labels share the high half a), Jb by counting, per popcount, the low halves seen so far
    const int h = N / 2, g = N - h;
    c->lin_h = h;
    std::vector<uint64_t> Ja((size_t)1 << g);
    std::vector<uint32_t> Jb((size_t)1 << h);
    uint64_t run = 0;
    for (uint64_t a = 0; a < (1ull << g); ++a) {
      Ja[(size_t)a] = run;
      run += binom_u64(h, N_up - __builtin_popcountll(a));
    }
    std::vector<uint32_t> seen((size_t)h + 1, 0);
    for (uint64_t b = 0; b < (1ull << h); ++b) Jb[(size_t)b] = seen[(size_t)__builtin_popcountll(b)]++;
    CKF(ftlm_dmalloc(&c->d_lin_hi, Ja.size() * 8));
    CKF(ftlm_dmalloc(&c->d_lin_lo, Jb.size() * 4));
    CKF(cudaMemcpy(c->d_lin_hi, Ja.data(), Ja.size() * 8, cudaMemcpyHostToDevice));
    CKF(cudaMemcpy(c->d_lin_lo, Jb.data(), Jb.size() * 4, cudaMemcpyHostToDevice));
  }
  for (int k = 0; k < 4; ++k) CKF(cudaEventCreate(&c->ev[k]));
  rc = ftlm_tml_plan_create(c);
  if (rc != FTLM_OK) return fail(rc);
  CKF(cudaDeviceSynchronize());
#undef CKF
  *out = c;
  return FTLM_OK;
}

extern "C" int ftlm_destroy(ftlm_ctx* c) {
  if (!c) return FTLM_OK;
  cudaSetDevice(c->device);
  graph_drop(c);
#ifndef FTLM_EMU
  if (c->graph_stream) cudaStreamDestroy((cudaStream_t)c->graph_stream);
#endif
  ftlm_tml_plan_destroy(c);
  ftlm_dfree(c->d_binom64); ftlm_dfree(c->d_binom32); ftlm_dfree(c->d_bonds); ftlm_dfree(c->d_clt);
  ftlm_dfree(c->d_state); ftlm_dfree(c->d_partials); ftlm_dfree(c->d_ticket); ftlm_dfree(c->d_lin_hi); ftlm_dfree(c->d_lin_lo);
  for (int k = 0; k < 3; ++k) ftlm_dfree(c->q[k]);
  for (int k = 0; k < 4; ++k) if (c->ev[k]) cudaEventDestroy(c->ev[k]);
  delete c;
  return FTLM_OK;
}

extern "C" int64_t ftlm_dim(const ftlm_ctx* c) { return c ? c->dim : -1; }

extern "C" int64_t ftlm_table_bytes(const ftlm_ctx* c) {
  if (!c) return -1;
  int64_t b = (int64_t)c->binom64.size() * 12 + (int64_t)c->nb * (int64_t)sizeof(BondDev);
  if (c->mode == FTLM_INDEX_CLT) b += c->n_clt * 8;
  if (c->mode == FTLM_INDEX_LIN) b += ((int64_t)8 << (c->N - c->lin_h)) + ((int64_t)4 << c->lin_h);
  return b;
}

int ftlm_effective_kernel(const ftlm_ctx* c) {
  if (c->kernel == FTLM_KERNEL_ROWG) return FTLM_KERNEL_ROWG;
  if (c->kernel == FTLM_KERNEL_ROW || c->mode == FTLM_INDEX_LIN) return FTLM_KERNEL_ROW;   // LIN: thread-per-row kernels only
  if (c->kernel == FTLM_KERNEL_TML && c->tml) return FTLM_KERNEL_TML;
  if (c->kernel == FTLM_KERNEL_AUTO && c->tml && c->dim >= (1 << 20)) return FTLM_KERNEL_TML;
  return FTLM_KERNEL_ROW;                    // AUTO: small sectors are launch-bound, ROW is simpler
}

extern "C" int ftlm_set_option(ftlm_ctx* c, const char* key, int64_t value) {
  if (!c || !key) { ftlm_set_error("ftlm_set_option: NULL"); return FTLM_EINVAL; }
  graph_drop(c);                                         // a captured step belongs to the configuration it was captured under
  if (!strcmp(key, "kernel")) {
    if (value != FTLM_KERNEL_AUTO && value != FTLM_KERNEL_ROW && value != FTLM_KERNEL_ROWG && value != FTLM_KERNEL_TML) { ftlm_set_error("kernel must be FTLM_KERNEL_AUTO, _ROW, _ROWG or _TML"); return FTLM_EINVAL; }
    if (value == FTLM_KERNEL_TML && (!c->tml || c->mode == FTLM_INDEX_LIN)) { ftlm_set_error("TML kernel unavailable for this sector / index mode"); return FTLM_EUNSUPPORTED; }
    c->kernel = (int)value; return FTLM_OK;
  }
  if (!strcmp(key, "tml_low_bits") || !strcmp(key, "tml_mid_bits")) {
    if (value < 0 || value > 16) { ftlm_set_error("%s must be 0..16", key); return FTLM_EINVAL; }
    int* slot = !strcmp(key, "tml_low_bits") ? &c->tml_low_bits : &c->tml_mid_bits;
    const int old = *slot;
    *slot = (int)value;
    CK(cudaSetDevice(c->device));
    ftlm_tml_plan_destroy(c);
    int rc = ftlm_tml_plan_create(c);
    if (rc != FTLM_OK) { *slot = old; ftlm_tml_plan_destroy(c); ftlm_tml_plan_create(c); }
    return rc;
  }
  if (!strcmp(key, "graph")) { c->use_graph = value ? 1 : 0; c->graph_failed = 0; return FTLM_OK; }
  if (!strcmp(key, "persistent")) { c->use_persistent = value ? 1 : 0; return FTLM_OK; }
  if (!strcmp(key, "allow_unverified")) { c->allow_unverified = value ? 1 : 0; return FTLM_OK; }
  if (!strcmp(key, "tmlr")) { c->use_tmlr = value ? 1 : 0; return FTLM_OK; }
  if (!strcmp(key, "lazy_norm")) { c->lazy_norm = value ? 1 : 0; return FTLM_OK; }
  if (!strcmp(key, "tmlr_unij")) {
    c->unij_allowed = value ? 1 : 0;
    CK(cudaSetDevice(c->device));
    ftlm_tml_plan_destroy(c);
    return ftlm_tml_plan_create(c);
  }
#if defined(FTLM_EMU) || defined(FTLM_CHECKED)
  // test hooks of the host-emulation and checked builds only (sampled tiles / items of full-size sectors);
  // the release library answers FTLM_EINVAL "unknown key"
  if (!strcmp(key, "debug_pass_mask")) { c->debug_pass_mask = (int)value; return FTLM_OK; }
  if (!strcmp(key, "debug_item_first")) { c->debug_item_first = value; return FTLM_OK; }
  if (!strcmp(key, "debug_item_count")) { c->debug_item_count = value; return FTLM_OK; }
#endif
  if (!strcmp(key, "autotune_mask")) { c->autotune_mask = (uint64_t)value; return FTLM_OK; }
  if (!strcmp(key, "batch") || !strcmp(key, "plan_batch")) {
    // "batch": chains per row pass of ftlm_lanczos / ftlm_lanczos_host (L207, L309); the TML split and the window
    // sizes are re-chosen so that tiles of `batch` interleaved vectors fit shared memory.  "plan_batch" (0 = follow
    // "batch"): build the plans for this many chains even when fewer run (same tiles and windows, hence the same
    // order of every sum: a chain then has bit-identical coefficients alone and inside a batch).
    const bool is_plan = key[0] == 'p';
    if (!(value == 1 || value == 2 || value == 4 || (is_plan && value == 0))) { ftlm_set_error("%s must be 1, 2 or 4", key); return FTLM_EINVAL; }
    int* slot = is_plan ? &c->plan_batch : &c->batch;
    const int old = *slot;
    *slot = (int)value;
    CK(cudaSetDevice(c->device));
    ftlm_tml_plan_destroy(c);
    int rc = ftlm_tml_plan_create(c);
    if (rc != FTLM_OK) { *slot = old; ftlm_tml_plan_destroy(c); ftlm_tml_plan_create(c); }
    return rc;
  }
  if (!strcmp(key, "passb") || !strcmp(key, "tml_split")) {
    // "passb": 0/1;  "tml_split": w | m << 8 (both at once; 0 = auto).  Rebuilds the TML / PASS-B plans.
    const int old_pb = c->use_passb, old_w = c->tml_low_bits, old_m = c->tml_mid_bits;
    if (!strcmp(key, "passb")) c->use_passb = value ? 1 : 0;
    else {
      if (value < 0 || (value & 0xff) > 16 || (value >> 8) > 16) { ftlm_set_error("tml_split must be w | m << 8"); return FTLM_EINVAL; }
      c->tml_low_bits = (int)(value & 0xff); c->tml_mid_bits = (int)(value >> 8);
    }
    CK(cudaSetDevice(c->device));
    ftlm_tml_plan_destroy(c);
    int rc = ftlm_tml_plan_create(c);
    if (rc != FTLM_OK) {
      c->use_passb = old_pb; c->tml_low_bits = old_w; c->tml_mid_bits = old_m;
      ftlm_tml_plan_destroy(c); ftlm_tml_plan_create(c);
    }
    return rc;
  }
  if (!strcmp(key, "passb_lo_min") || !strcmp(key, "passb_smax") || !strcmp(key, "passb_ctas")) {
    // PASS-B window planner knobs (0 = auto); rebuilds the TML / PASS-B plans
    if (value < 0 || value > 62) { ftlm_set_error("%s out of range", key); return FTLM_EINVAL; }
    int* slot = !strcmp(key, "passb_lo_min") ? &c->passb_lo_min : !strcmp(key, "passb_smax") ? &c->passb_smax : &c->passb_ctas;
    const int old = *slot;
    *slot = (int)value;
    CK(cudaSetDevice(c->device));
    ftlm_tml_plan_destroy(c);
    int rc = ftlm_tml_plan_create(c);
    if (rc != FTLM_OK) { *slot = old; ftlm_tml_plan_destroy(c); ftlm_tml_plan_create(c); }
    return rc;
  }
  ftlm_set_error("ftlm_set_option: unknown key '%s'", key);
  return FTLM_EINVAL;
}

extern "C" int64_t ftlm_get_option(const ftlm_ctx* c, const char* key) {
  if (!key) return -1;
  if (!strncmp(key, "check_", 6)) {                      // checked build (ftlm_access.cuh): process-wide, ctx may be NULL
#if defined(FTLM_CHECKED) && !defined(FTLM_EMU)
    if (!strcmp(key, "check_build")) return 1;
    return chk_read(key);
#else
    return !strcmp(key, "check_build") ? 0 : -1;
#endif
  }
  if (!c) return -1;
  if (!strcmp(key, "kernel")) return ftlm_effective_kernel(c);
  if (!strcmp(key, "graph")) return c->use_graph;
  if (!strcmp(key, "persistent")) return c->use_persistent;
  if (!strcmp(key, "persistent_fits")) return ftlm_chain_persistent_fits(c) ? 1 : 0;
  if (!strcmp(key, "graph_launches")) return c->graph_launches;
  if (!strcmp(key, "graph_failed")) return c->graph_failed;
  if (!strcmp(key, "passb")) return c->use_passb;
  if (!strncmp(key, "passb_", 6)) return ftlm_passb_info(c, key);
  if (!strcmp(key, "sm_count")) return c->sm_count;
  if (!strcmp(key, "autotuned")) return c->autotuned;
  if (!strcmp(key, "allow_unverified")) return c->allow_unverified;
  if (!strcmp(key, "autotune_mask")) return (int64_t)c->autotune_mask;
  if (!strcmp(key, "batch")) return c->batch;
  if (!strcmp(key, "plan_batch")) return c->plan_batch;
  if (!strcmp(key, "tmlr")) return c->use_tmlr;
  if (!strcmp(key, "lazy_norm")) return c->lazy_norm;
  if (!strcmp(key, "lazy_norm_ok")) return ftlm_tmlr_lazy_ok(c) ? 1 : 0;
  if (!strncmp(key, "tmlr_", 5)) return ftlm_tmlr_info(c, key);
  if (!strncmp(key, "tml_", 4)) return ftlm_tml_info(c, key);
  return -1;
}

extern "C" int ftlm_clt_read(ftlm_ctx* c, int64_t b0, int64_t nb, uint32_t* h_mask, uint32_t* h_count) {
  if (!c || c->mode != FTLM_INDEX_CLT || b0 < 0 || nb < 0 || b0 + nb > c->n_clt || !h_mask || !h_count) {
    ftlm_set_error("ftlm_clt_read: bad argument or not a CLT handle"); return FTLM_EINVAL;
  }
  CK(cudaSetDevice(c->device));
  std::vector<uint2> tmp((size_t)nb);
  CK(cudaMemcpy(tmp.data(), c->d_clt + b0, sizeof(uint2) * (size_t)nb, cudaMemcpyDeviceToHost));
  for (int64_t k = 0; k < nb; ++k) { h_mask[k] = tmp[(size_t)k].x; h_count[k] = tmp[(size_t)k].y; }
  return FTLM_OK;
}

// ---- H.v ---------------------------------------------------------------------------------------
static int launch_hv(ftlm_ctx* c, const void* v, const void* qp, void* y, int fused, cudaStream_t s, int batch = 1) {
  const int k = ftlm_effective_kernel(c);
  if (k == FTLM_KERNEL_TML) {
    // multi-pass step when PASS-B windows exist: the in-tile pass leaves the sums and the finish to the last window.
    // batch > 1 (L207): rows of `batch` interleaved chains through the same passes (TML in-tile pass; the
    // register-table TMLR pass is a single-vector kernel)
    const bool pb = c->passb != nullptr;
    int rc = FTLM_OK;
    if (batch > ftlm_plan_batch(c)) { ftlm_set_error("batch %d: the plans of this handle were built for %d chains (option \"batch\")", batch, ftlm_plan_batch(c)); return FTLM_EINVAL; }
    if (fused || !c->debug_pass_mask || (c->debug_pass_mask & 1)) {
      if (c->use_tmlr && c->tmlr && batch == 1) rc = ftlm_launch_hv_tmlr(c, v, qp, y, fused ? (pb ? 2 : 1) : 0, s);
      else rc = ftlm_launch_hv_tml(c, v, qp, y, fused ? (pb ? 2 : 1) : 0, batch, s);
    }
    if (rc == FTLM_OK && pb) rc = ftlm_launch_passb(c, v, y, fused, batch, s);
    return rc;
  }
  if (k == FTLM_KERNEL_ROWG && batch == 1) return ftlm_launch_hv_rowg(c, v, qp, y, fused, s);   // (a batch runs the ROW kernel)
  return ftlm_launch_hv_row(c, v, qp, y, fused, batch, s);
}

extern "C" int ftlm_apply_H(ftlm_ctx* c, const void* d_v, void* d_y, void* stream) {
  if (!c || !d_v || !d_y || d_v == d_y) { ftlm_set_error("ftlm_apply_H: bad argument (NULL or d_y == d_v)"); return FTLM_EINVAL; }
  CK(cudaSetDevice(c->device));
  ftlm_chk_caller((cudaStream_t)stream, d_v, (size_t)c->dim * ftlm_elem_size(c));
  ftlm_chk_caller((cudaStream_t)stream, d_y, (size_t)c->dim * ftlm_elem_size(c));
  return launch_hv(c, d_v, nullptr, d_y, 0, (cudaStream_t)stream);
}

extern "C" int ftlm_apply_H_host(ftlm_ctx* c, const void* h_v, void* h_y) {
  if (!c || !h_v || !h_y) { ftlm_set_error("ftlm_apply_H_host: NULL"); return FTLM_EINVAL; }
  CK(cudaSetDevice(c->device));
  const size_t bytes = (size_t)c->dim * ftlm_elem_size(c);
  void *dv = nullptr, *dy = nullptr;
  if (ftlm_dmalloc(&dv, bytes) != cudaSuccess || ftlm_dmalloc(&dy, bytes) != cudaSuccess) {
    ftlm_dfree(dv); ftlm_set_error("ftlm_apply_H_host: out of device memory"); return FTLM_ENOMEM;
  }
  int rc = FTLM_OK;
  cudaError_t e = cudaMemcpy(dv, h_v, bytes, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) rc = launch_hv(c, dv, nullptr, dy, 0, 0);
  if (e == cudaSuccess && rc == FTLM_OK) e = cudaMemcpy(h_y, dy, bytes, cudaMemcpyDeviceToHost);
  ftlm_dfree(dv); ftlm_dfree(dy);
  if (e != cudaSuccess) return ftlm_cuda_fail(e, "ftlm_apply_H_host");
  return rc;
}

extern "C" int ftlm_neighbors(ftlm_ctx* c, int64_t row0, int64_t nrows, int64_t* d_idx, void* stream) {
  if (!c || row0 < 0 || nrows < 0 || row0 + nrows > c->dim || (nrows > 0 && !d_idx)) {
    ftlm_set_error("ftlm_neighbors: bad row range"); return FTLM_EINVAL;
  }
  if (nrows == 0 || c->nb == 0) return FTLM_OK;
  CK(cudaSetDevice(c->device));
  ftlm_chk_caller((cudaStream_t)stream, d_idx, (size_t)nrows * (size_t)c->nb * 8);
  if (ftlm_effective_kernel(c) == FTLM_KERNEL_TML) return ftlm_launch_neighbors_tml(c, row0, nrows, d_idx, (cudaStream_t)stream);
  if (ftlm_effective_kernel(c) == FTLM_KERNEL_ROWG) return ftlm_launch_neighbors_rowg(c, row0, nrows, d_idx, (cudaStream_t)stream);
  return ftlm_launch_neighbors_row(c, row0, nrows, d_idx, (cudaStream_t)stream);
}

// ---- start vectors -----------------------------------------------------------------------------
uint64_t ftlm_chain_key(uint64_t seed, int N_up, int r);
static uint64_t chain_key(uint64_t seed, int N_up, int r) { return ftlm_chain_key(seed, N_up, r); }
uint64_t ftlm_chain_key(uint64_t seed, int N_up, int r) {
  uint64_t k = mix64_host(seed);
  k = mix64_host(k + FTLM_GOLD * (uint64_t)(N_up + 1));
  k = mix64_host(k + FTLM_GOLD * (uint64_t)(r + 1));
  return k;
}

static int stream_grid(const ftlm_ctx* c, int64_t n, int per_sm) {
  int64_t blocks = (n + 255) / 256;
  int64_t cap = (int64_t)c->sm_count * per_sm;
  if (blocks > cap) blocks = cap;
  if (blocks > c->max_blocks) blocks = c->max_blocks;
  return (int)(blocks < 1 ? 1 : blocks);
}

extern "C" int ftlm_fill_random(ftlm_ctx* c, uint64_t seed, int r, void* d_v, void* stream) {
  if (!c || !d_v || r < 0) { ftlm_set_error("ftlm_fill_random: bad argument"); return FTLM_EINVAL; }
  CK(cudaSetDevice(c->device));
  cudaStream_t s = (cudaStream_t)stream;
  ftlm_chk_caller(s, d_v, (size_t)c->dim * ftlm_elem_size(c));
  const uint64_t key = chain_key(seed, c->N_up, r);
  const int grid = stream_grid(c, c->dim, 8);
  FTLM_LAUNCH(gauss_norm_kernel, grid, 256, 0, s, key, c->dim, c->d_partials);
  FTLM_LAUNCH(reduce_partials_kernel, 1, 256, 0, s, c->d_partials, grid, &c->d_state->norm2);
  if (c->prec == FTLM_FP32) { auto k__ = gauss_write_kernel<float>; FTLM_LAUNCH(k__, grid, 256, 0, s, key, c->dim, &c->d_state->norm2, (float*)d_v, 1, 0); }
  else { auto k__ = gauss_write_kernel<double>; FTLM_LAUNCH(k__, grid, 256, 0, s, key, c->dim, &c->d_state->norm2, (double*)d_v, 1, 0); }
  CK(cudaGetLastError());
  return FTLM_OK;
}

// ---- chain -------------------------------------------------------------------------------------
static int ensure_workspace(ftlm_ctx* c, int batch) {
  const size_t bytes = (size_t)c->dim * ftlm_elem_size(c) * (size_t)batch;
  if (c->q_batch < batch) {                            // (re)allocate for the widest batch seen so far
    for (int k = 0; k < 3; ++k) { ftlm_dfree(c->q[k]); c->q[k] = nullptr; }
    c->q_batch = 0;
  }
  for (int k = 0; k < 3; ++k)
    if (!c->q[k]) {
      cudaError_t e = ftlm_dmalloc(&c->q[k], bytes);
      if (e != cudaSuccess) { ftlm_set_error("chain workspace: cannot allocate 3 x %zu bytes (%s)", bytes, cudaGetErrorString(e)); cudaGetLastError(); return FTLM_ENOMEM; }
    }
  if (c->q_batch < batch) c->q_batch = batch;
  return FTLM_OK;
}

// Begin `batch` chains r0 .. r0 + batch - 1 on interleaved work vectors q[t][batch] (batch = 1: plain vectors).
// q1 == nullptr: seeded start vectors; else `batch` vectors of dim elements each, one after the other.
static int chain_begin_impl(ftlm_ctx* c, const void* q1, bool q1_on_host, uint64_t seed, int r0, int batch, cudaStream_t s) {
  CK(cudaSetDevice(c->device));
  if (batch != 1 && batch != 2 && batch != 4) { ftlm_set_error("batch must be 1, 2 or 4 (got %d)", batch); return FTLM_EINVAL; }
  int rc = ensure_workspace(c, batch);
  if (rc != FTLM_OK) return rc;
  const size_t vbytes = (size_t)c->dim * ftlm_elem_size(c), bytes = vbytes * (size_t)batch;
  c->ia = 0; c->ib = 1; c->ic = 2;
  c->pending_norm = false;
  c->steps_enqueued = 0;
  c->cur_batch = batch;
  c->chain_limit = (int)(c->dim < FTLM_MAX_STEPS ? c->dim : FTLM_MAX_STEPS);
  const int grid = stream_grid(c, c->dim, 8);
  for (int b = 0; b < batch; ++b) {
    double* norm2 = &c->d_state[b].norm2;
    if (!q1) {
      const uint64_t key = chain_key(seed, c->N_up, r0 + b);
      FTLM_LAUNCH(gauss_norm_kernel, grid, 256, 0, s, key, c->dim, c->d_partials);
      FTLM_LAUNCH(reduce_partials_kernel, 1, 256, 0, s, c->d_partials, grid, norm2);
      if (c->prec == FTLM_FP32) { auto k__ = gauss_write_kernel<float>; FTLM_LAUNCH(k__, grid, 256, 0, s, key, c->dim, norm2, (float*)c->q[0], batch, b); }
      else { auto k__ = gauss_write_kernel<double>; FTLM_LAUNCH(k__, grid, 256, 0, s, key, c->dim, norm2, (double*)c->q[0], batch, b); }
    } else {
      // copy into q[2] (scratch), then normalise in FP64 into column b of q[0]
      CK(cudaMemcpyAsync(c->q[2], (const char*)q1 + (size_t)b * vbytes, vbytes, q1_on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, s));
      if (c->prec == FTLM_FP32) { auto k__ = sumsq_kernel<float>; FTLM_LAUNCH(k__, grid, 256, 0, s, (const float*)c->q[2], c->dim, c->d_partials); }
      else { auto k__ = sumsq_kernel<double>; FTLM_LAUNCH(k__, grid, 256, 0, s, (const double*)c->q[2], c->dim, c->d_partials); }
      FTLM_LAUNCH(reduce_partials_kernel, 1, 256, 0, s, c->d_partials, grid, norm2);
      if (c->prec == FTLM_FP32) { auto k__ = scale_copy_kernel<float>; FTLM_LAUNCH(k__, grid, 256, 0, s, (const float*)c->q[2], c->dim, norm2, (float*)c->q[0], batch, b); }
      else { auto k__ = scale_copy_kernel<double>; FTLM_LAUNCH(k__, grid, 256, 0, s, (const double*)c->q[2], c->dim, norm2, (double*)c->q[0], batch, b); }
    }
  }
  CK(cudaMemsetAsync(c->q[1], 0, bytes, s));          // q_0 = 0
  FTLM_LAUNCH(chain_reset_kernel, 1, 32, 0, s, c->d_state, c->chain_limit, c->prec == FTLM_FP32 ? 1e-5 : 1e-12, batch);
  CK(cudaGetLastError());
  return FTLM_OK;
}

extern "C" int ftlm_chain_begin(ftlm_ctx* c, const void* d_q1, uint64_t seed, int r, void* stream) {
  if (!c || r < 0) { ftlm_set_error("ftlm_chain_begin: bad argument"); return FTLM_EINVAL; }
  if (d_q1) ftlm_chk_caller((cudaStream_t)stream, d_q1, (size_t)c->dim * ftlm_elem_size(c));
  return chain_begin_impl(c, d_q1, false, seed, r, 1, (cudaStream_t)stream);
}

static int launch_next(ftlm_ctx* c, cudaStream_t s) {
  const void* y = c->q[c->ic];
  const void* q = c->q[c->ia];
  void* qn = c->q[c->ib];
  const int64_t n = c->dim * c->cur_batch;             // interleaved batch: element i belongs to chain i % batch
  const int grid = stream_grid(c, n / 4 + 1, 8);
#define NEXT(BB)                                                                                                     \
  do {                                                                                                               \
    if (c->prec == FTLM_FP32) { auto k__ = lanczos_next_kernel<float, float4, BB>; FTLM_LAUNCH(k__, grid, 256, 0, s, (const float*)y, (const float*)q, (float*)qn, n, c->d_state); } \
    else { auto k__ = lanczos_next_kernel<double, double2, BB>; FTLM_LAUNCH(k__, grid, 256, 0, s, (const double*)y, (const double*)q, (double*)qn, n, c->d_state); } \
  } while (0)
  if (c->cur_batch == 1) NEXT(1); else if (c->cur_batch == 2) NEXT(2); else NEXT(4);
#undef NEXT
  CK(cudaGetLastError());
  return FTLM_OK;
}

static int chain_one_step(ftlm_ctx* c, cudaStream_t s, bool timed, float* ms_hv, float* ms_norm) {
  // lazy normalisation (option "lazy_norm", TMLR in-tile pass only): no normalisation pass; the next step's
  // in-tile pass forms q_{j+1} = (y_j - alpha_j q_j)/beta_j while it stages its tile and writes it over y_j
  const bool lazy = c->cur_batch == 1 && c->lazy_norm && ftlm_effective_kernel(c) == FTLM_KERNEL_TML && ftlm_tmlr_lazy_ok(c);
  // y = H q_j - beta_{j-1} q_{j-1}   (+ reductions, alpha_j, beta_j on the device)
  if (timed) CK(cudaEventRecord(c->ev[0], s));
  int rc;
  if (lazy && c->pending_norm) {
    const bool pb = c->passb != nullptr;
    rc = ftlm_launch_hv_tmlr_lazy(c, c->q[c->ic], c->q[c->ia], c->q[c->ib], pb ? 2 : 1, s);
    if (rc == FTLM_OK && pb) rc = ftlm_launch_passb(c, c->q[c->ic], c->q[c->ib], 1, 1, s);
    const int a = c->ia, b = c->ib, y = c->ic;             // q_{j+1} now lives in the old y, q_j becomes q_prev, y is the old q_{j-1}
    c->ia = y; c->ib = a; c->ic = b;
  } else {
    if (c->pending_norm) {                                 // the option was switched off mid-chain: materialise q_{j+1} first
      rc = launch_next(c, s);
      if (rc != FTLM_OK) return rc;
      const int a = c->ia; c->ia = c->ib; c->ib = a;
      c->pending_norm = false;
    }
    rc = launch_hv(c, c->q[c->ia], c->q[c->ib], c->q[c->ic], 1, s, c->cur_batch);
  }
  if (rc != FTLM_OK) return rc;
  if (timed) CK(cudaEventRecord(c->ev[1], s));
  if (lazy) c->pending_norm = true;
  else {
    // q_{j+1} = (y - alpha_j q_j)/beta_j, written over q_{j-1}; then q_{j+1} <-> q_j roles swap, y stays
    rc = launch_next(c, s);
    if (rc != FTLM_OK) return rc;
    const int a = c->ia; c->ia = c->ib; c->ib = a;
  }
  if (timed) {
    CK(cudaEventRecord(c->ev[2], s));
    CK(cudaEventSynchronize(c->ev[2]));
    CK(cudaEventElapsedTime(ms_hv, c->ev[0], c->ev[1]));
    CK(cudaEventElapsedTime(ms_norm, c->ev[1], c->ev[2]));
  }
  c->steps_enqueued++;
  return FTLM_OK;
}

// ---- CUDA graph of the step (option "graph"; SURVEY 3(i), 8(d) "CUDA events around a graph of N_L steps") -------------
// The work-vector roles return to where they were after `period` steps (2: q_j / q_{j-1} swap; 3 with lazy
// normalisation), so `period` consecutive steps are captured once and replayed.  Breakdown stays a device-side no-op.
// Any failure of a graph call leaves the handle on direct launches (never an error of the chain).
static void graph_drop(ftlm_ctx* c) {
#ifndef FTLM_EMU
  if (c->graph_exec) { cudaGraphExecDestroy((cudaGraphExec_t)c->graph_exec); c->graph_exec = nullptr; }
#endif
  c->graph_roles[0] = c->graph_roles[1] = c->graph_roles[2] = -1;
}

#ifndef FTLM_EMU
static bool graph_ready(ftlm_ctx* c, int period) {
  if (c->graph_exec && c->graph_roles[0] == c->ia && c->graph_roles[1] == c->ib && c->graph_roles[2] == c->ic &&
      c->graph_batch == c->cur_batch && c->graph_period == period) return true;
  graph_drop(c);
  if (!c->graph_stream) {
    cudaStream_t gs = nullptr;
    if (cudaStreamCreateWithFlags(&gs, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); c->graph_failed = 1; return false; }
    c->graph_stream = gs;
  }
  cudaStream_t gs = (cudaStream_t)c->graph_stream;
  const int ia = c->ia, ib = c->ib, ic = c->ic, enq = c->steps_enqueued;
  const bool pend = c->pending_norm;
  cudaGraph_t g = nullptr;
  bool ok = cudaStreamBeginCapture(gs, cudaStreamCaptureModeRelaxed) == cudaSuccess;
  if (ok) {
    for (int k = 0; k < period && ok; ++k) ok = chain_one_step(c, gs, false, nullptr, nullptr) == FTLM_OK;
    ok = (cudaStreamEndCapture(gs, &g) == cudaSuccess) && ok && g != nullptr;
  }
  ok = ok && c->ia == ia && c->ib == ib && c->ic == ic && c->pending_norm == pend;   // the roles are periodic
  c->ia = ia; c->ib = ib; c->ic = ic; c->steps_enqueued = enq; c->pending_norm = pend;  // nothing has run
  cudaGraphExec_t ge = nullptr;
  if (ok) ok = cudaGraphInstantiate(&ge, g, 0) == cudaSuccess;
  if (g) cudaGraphDestroy(g);
  if (!ok) { cudaGetLastError(); c->graph_failed = 1; return false; }
  c->graph_exec = ge;
  c->graph_roles[0] = ia; c->graph_roles[1] = ib; c->graph_roles[2] = ic;
  c->graph_batch = c->cur_batch; c->graph_period = period;
  return true;
}
#endif

extern "C" int ftlm_chain_steps(ftlm_ctx* c, int nsteps, void* stream) {
  if (!c || nsteps < 0 || !c->q[0]) { ftlm_set_error("ftlm_chain_steps: no chain begun or nsteps < 0"); return FTLM_EINVAL; }
  CK(cudaSetDevice(c->device));
  int k = 0;
#ifndef FTLM_EMU
  if (c->use_graph && !c->graph_failed) {
    const bool lazy = c->cur_batch == 1 && c->lazy_norm && ftlm_effective_kernel(c) == FTLM_KERNEL_TML && ftlm_tmlr_lazy_ok(c);
    const int period = lazy ? 3 : 2;
    // the first step of a chain runs directly (lazy form: it is the one step without a pending normalisation)
    for (; k < nsteps && c->steps_enqueued < 1 && c->steps_enqueued < c->chain_limit; ++k) {
      int rc = chain_one_step(c, (cudaStream_t)stream, false, nullptr, nullptr);
      if (rc != FTLM_OK) return rc;
    }
    while (nsteps - k >= period && c->steps_enqueued + period <= c->chain_limit && graph_ready(c, period)) {
      if (cudaGraphLaunch((cudaGraphExec_t)c->graph_exec, (cudaStream_t)stream) != cudaSuccess) { cudaGetLastError(); c->graph_failed = 1; break; }
      c->steps_enqueued += period;
      c->graph_launches++;
      k += period;
    }
  }
#endif
  for (; k < nsteps; ++k) {
    if (c->steps_enqueued >= c->chain_limit) break;      // the device would no-op anyway
    int rc = chain_one_step(c, (cudaStream_t)stream, false, nullptr, nullptr);
    if (rc != FTLM_OK) return rc;
  }
  return FTLM_OK;
}

extern "C" int ftlm_chain_profile(ftlm_ctx* c, int nsteps, void* stream, double* ms_hv, double* ms_norm) {
  if (!c || nsteps <= 0 || !c->q[0] || !ms_hv || !ms_norm) { ftlm_set_error("ftlm_chain_profile: bad argument"); return FTLM_EINVAL; }
  CK(cudaSetDevice(c->device));
  double a = 0.0, b = 0.0;
  int n = 0;
  for (int k = 0; k < nsteps; ++k) {
    if (c->steps_enqueued >= c->chain_limit) break;
    float x = 0.f, y = 0.f;
    int rc = chain_one_step(c, (cudaStream_t)stream, true, &x, &y);
    if (rc != FTLM_OK) return rc;
    a += x; b += y; ++n;
  }
  *ms_hv = n ? a / n : 0.0;
  *ms_norm = n ? b / n : 0.0;
  return FTLM_OK;
}

// coefficients of chain b of the batch in progress: alpha -> h_alpha + b * cap, beta -> h_beta + b * cap
static int chain_end_impl(ftlm_ctx* c, double* h_alpha, double* h_beta, int cap, int* h_m_eff, int batch, cudaStream_t s) {
  CK(cudaSetDevice(c->device));
  CK(cudaStreamSynchronize(s));
  static thread_local ChainState hs[FTLM_MAX_BATCH];
  CK(cudaMemcpy(hs, c->d_state, sizeof(ChainState) * (size_t)batch, cudaMemcpyDeviceToHost));
  for (int b = 0; b < batch; ++b) {
    int m = hs[b].step;
    h_m_eff[b] = m;
    if (m > cap) m = cap;
    if (h_alpha) for (int k = 0; k < m; ++k) h_alpha[(size_t)b * cap + k] = hs[b].alpha[k];
    if (h_beta) for (int k = 0; k + 1 < m; ++k) h_beta[(size_t)b * cap + k] = hs[b].beta[k];
  }
  return FTLM_OK;
}

extern "C" int ftlm_chain_end(ftlm_ctx* c, double* h_alpha, double* h_beta, int cap, int* h_m_eff, void* stream) {
  if (!c || !h_m_eff || cap < 0) { ftlm_set_error("ftlm_chain_end: bad argument"); return FTLM_EINVAL; }
  if (c->cur_batch != 1) { ftlm_set_error("ftlm_chain_end: a batch of %d chains is in progress; use ftlm_chain_end_batch", c->cur_batch); return FTLM_EINVAL; }
  return chain_end_impl(c, h_alpha, h_beta, cap, h_m_eff, 1, (cudaStream_t)stream);
}

extern "C" int ftlm_chain_begin_batch(ftlm_ctx* c, uint64_t seed, int r0, int batch, void* stream) {
  if (!c || r0 < 0) { ftlm_set_error("ftlm_chain_begin_batch: bad argument"); return FTLM_EINVAL; }
  return chain_begin_impl(c, nullptr, false, seed, r0, batch, (cudaStream_t)stream);
}

extern "C" int ftlm_chain_end_batch(ftlm_ctx* c, double* h_alpha, double* h_beta, int cap, int* h_m_eff, void* stream) {
  if (!c || !h_m_eff || cap < 0) { ftlm_set_error("ftlm_chain_end_batch: bad argument"); return FTLM_EINVAL; }
  return chain_end_impl(c, h_alpha, h_beta, cap, h_m_eff, c->cur_batch, (cudaStream_t)stream);
}

static int lanczos_impl(ftlm_ctx* c, const void* h_q1, uint64_t seed, int R, int n_steps, double* h_alpha,
                        double* h_beta, int* h_m_eff, double* h_theta, double* h_weight, cudaStream_t s) {
  if (!c || R < 0 || n_steps < 1 || n_steps > FTLM_MAX_STEPS || !h_alpha || !h_beta || !h_m_eff) {
    ftlm_set_error("ftlm_lanczos: bad argument (n_steps must be in [1,%d])", FTLM_MAX_STEPS); return FTLM_EINVAL;
  }
  const size_t bytes = (size_t)c->dim * ftlm_elem_size(c);
  for (size_t k = 0; k < (size_t)R * n_steps; ++k) { h_alpha[k] = 0.0; h_beta[k] = 0.0; }
  if (c->use_persistent && !h_q1 && R > 0 && ftlm_chain_persistent_fits(c)) {
    // small sector: all R chains in ONE launch, one CTA per chain, vectors in shared memory (ftlm_chain.cu)
    CK(cudaSetDevice(c->device));
    const int limit = (int)std::min<int64_t>(n_steps, c->dim);
    double *d_a = nullptr, *d_b = nullptr;
    int* d_m = nullptr;
    const size_t nb = (size_t)R * limit * 8;
    if (ftlm_dmalloc(&d_a, nb) != cudaSuccess || ftlm_dmalloc(&d_b, nb) != cudaSuccess || ftlm_dmalloc(&d_m, (size_t)R * 4) != cudaSuccess) {
      cudaGetLastError(); ftlm_dfree(d_a); ftlm_dfree(d_b); ftlm_dfree(d_m);
      ftlm_set_error("ftlm_lanczos: out of device memory"); return FTLM_ENOMEM;
    }
    int rc = ftlm_launch_chain_persistent(c, seed, 0, R, limit, d_a, d_b, d_m, s);
    std::vector<double> ha((size_t)R * limit), hb((size_t)R * limit);
    if (rc == FTLM_OK && (cudaMemcpy(ha.data(), d_a, nb, cudaMemcpyDeviceToHost) != cudaSuccess || cudaMemcpy(hb.data(), d_b, nb, cudaMemcpyDeviceToHost) != cudaSuccess ||
                          cudaMemcpy(h_m_eff, d_m, (size_t)R * 4, cudaMemcpyDeviceToHost) != cudaSuccess))
      rc = ftlm_cuda_fail(cudaGetLastError(), "ftlm_lanczos: copy of the coefficients");
    ftlm_dfree(d_a); ftlm_dfree(d_b); ftlm_dfree(d_m);
    if (rc != FTLM_OK) return rc;
    for (int r = 0; r < R; ++r) {
      const int m = h_m_eff[r];
      for (int k = 0; k < m; ++k) h_alpha[(size_t)r * n_steps + k] = ha[(size_t)r * limit + k];
      for (int k = 0; k + 1 < m; ++k) h_beta[(size_t)r * n_steps + k] = hb[(size_t)r * limit + k];
      if (h_theta && h_weight) {
        double* th = h_theta + (size_t)r * n_steps;
        double* w = h_weight + (size_t)r * n_steps;
        for (int k = 0; k < n_steps; ++k) { th[k] = 0.0; w[k] = 0.0; }
        rc = ftlm_tridiag_eig(m, h_alpha + (size_t)r * n_steps, h_beta + (size_t)r * n_steps, th, w);
        if (rc != FTLM_OK) return rc;
      }
    }
    return FTLM_OK;
  }
  // chains advance in groups of option "batch" (4, 2 or 1) on interleaved vectors; a remainder runs in smaller groups
  for (int r = 0; r < R;) {
    int nb = c->batch;
    while (nb > R - r) nb >>= 1;
    double* a = h_alpha + (size_t)r * n_steps;
    double* b = h_beta + (size_t)r * n_steps;
    int rc = chain_begin_impl(c, h_q1 ? (const char*)h_q1 + (size_t)r * bytes : nullptr, h_q1 != nullptr, seed, r, nb, s);
    if (rc != FTLM_OK) return rc;
    if (c->chain_limit > n_steps) {           // m = min(n_steps, dim)
      c->chain_limit = n_steps;
      FTLM_LAUNCH(chain_reset_kernel, 1, 32, 0, s, c->d_state, n_steps, c->prec == FTLM_FP32 ? 1e-5 : 1e-12, nb);
    }
    rc = ftlm_chain_steps(c, n_steps, s);
    if (rc != FTLM_OK) return rc;
    rc = chain_end_impl(c, a, b, n_steps, &h_m_eff[r], nb, s);
    if (rc != FTLM_OK) return rc;
    if (h_theta && h_weight) {
      for (int q = 0; q < nb; ++q) {
        double* th = h_theta + (size_t)(r + q) * n_steps;
        double* w = h_weight + (size_t)(r + q) * n_steps;
        for (int k = 0; k < n_steps; ++k) { th[k] = 0.0; w[k] = 0.0; }
        rc = ftlm_tridiag_eig(h_m_eff[r + q], a + (size_t)q * n_steps, b + (size_t)q * n_steps, th, w);
        if (rc != FTLM_OK) return rc;
      }
    }
    r += nb;
  }
  c->cur_batch = 1;
  return FTLM_OK;
}

extern "C" int ftlm_lanczos(ftlm_ctx* c, uint64_t seed, int R, int n_steps, double* h_alpha, double* h_beta,
                            int* h_m_eff, double* h_theta, double* h_weight, void* stream) {
  return lanczos_impl(c, nullptr, seed, R, n_steps, h_alpha, h_beta, h_m_eff, h_theta, h_weight, (cudaStream_t)stream);
}

extern "C" int ftlm_lanczos_host(ftlm_ctx* c, const void* h_q1, int R, int n_steps, double* h_alpha, double* h_beta,
                                 int* h_m_eff, double* h_theta, double* h_weight, void* stream) {
  if (!h_q1) { ftlm_set_error("ftlm_lanczos_host: h_q1 is NULL"); return FTLM_EINVAL; }
  return lanczos_impl(c, h_q1, 0, R, n_steps, h_alpha, h_beta, h_m_eff, h_theta, h_weight, (cudaStream_t)stream);
}
