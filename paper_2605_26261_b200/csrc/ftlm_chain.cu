// Persistent chain kernel: whole Lanczos chains of a SMALL sector in one launch ("configs 1-2 are
// launch-bound ... use CUDA graphs or a persistent kernel, batch all R chains").
//
// One CTA owns one chain.  Its three work vectors q_j, q_{j-1}, y live in shared memory for the whole chain (3 D
// elements: D <= ~17 000 in FP32, ~8 500 in FP64 with 200 KB), so a step costs no global vector traffic and no
// launch: the start vector comes from the counter-based generator (FP64 norm), then per step
//   y = H q_j - beta_{j-1} q_{j-1}   row by row (thread-per-row form of Eq. 12: unrank, bond loop,
//                                     index by Alg. 2 / incremental Alg. 1 / Lin tables, gathers from shared memory),
//   alpha_j = <q,y>/<q,q>, beta_j^2 = <y,y> - <q,y>^2/<q,q>  (FP64 sums, fixed-order block reduction: reading 11, H9),
//   q_{j+1} = (y - alpha_j q_j)/beta_j   written over q_{j-1}; breakdown rule of reading 10.
// Same arithmetic as the fused ROW step + normalisation pass (vectors in the handle's precision, sums in FP64);
// only the order of the reduction differs.  grid = number of chains (all R chains of a sector in ONE launch).
#define FTLM_TU 7
#include "ftlm_common.cuh"
#include "ftlm_index.cuh"

#define CHAIN_THREADS 1024

namespace {

struct ChainParams {
  int N, K, nb, mode, limit;
  int labels;                // 1: the row labels are unranked once per chain and kept in shared memory (when they fit)
  int lin_h;
  const uint64_t* lin_hi;
  const uint32_t* lin_lo;
  int64_t dim;
  const void* binom;         // I[(N+1)*(K+1)]
  const BondDev* bonds;
  const uint2* clt;
  double diag0, tol;
  double* alpha;             // [nchains][limit]
  double* beta;              // [nchains][limit]
  int* m_eff;                // [nchains]
};

template <typename R> struct CBond { uint64_t mask; R Jh, Jq; int i, j; };

// lsz: bytes per stored row label (0 = labels are unranked on the fly every step)
__host__ __device__ inline size_t chain_smem_bytes(int N, int K, int nb, int64_t dim, int esz, int isz, int bond_sz, int lsz) {
  size_t o = ((size_t)(N + 1) * (K + 1) * isz + 15) & ~(size_t)15;
  o += ((size_t)nb * bond_sz + 15) & ~(size_t)15;
  o += (size_t)96 * 8 + 64;                              // reduction scratch + scalars
  o += 3 * (((size_t)dim * esz + 15) & ~(size_t)15);
  o += ((size_t)dim * lsz + 15) & ~(size_t)15;
  return o;
}

template <typename R, typename L, typename I, int MODE>
__global__ void __launch_bounds__(CHAIN_THREADS, 1)
lanczos_chain_kernel(ChainParams p, const uint64_t* __restrict__ keys) {
  FTLM_DYN_SMEM(smem);
  const int tid = threadIdx.x, NT = blockDim.x;
  const int K1 = p.K + 1, D = (int)p.dim;
  I* s_binom = (I*)smem;
  size_t o = ((size_t)(p.N + 1) * K1 * sizeof(I) + 15) & ~(size_t)15;
  CBond<R>* s_bonds = (CBond<R>*)(smem + o);
  o += ((size_t)p.nb * sizeof(CBond<R>) + 15) & ~(size_t)15;
  double* s_red = (double*)(smem + o);                     // [96] block_sum3 scratch
  double* s_sc = s_red + 96;                               // [0] beta_prev, [1] alpha, [2] 1/beta, [3] scale, [4] done flag, [5] norm
  o += (size_t)96 * 8 + 64;
  const size_t vstride = (((size_t)D * sizeof(R) + 15) & ~(size_t)15) / sizeof(R);
  R* vec = (R*)(smem + o);
  o += 3 * (((size_t)D * sizeof(R) + 15) & ~(size_t)15);
  L* lab = (L*)(smem + o);                                 // [D] row labels (only if p.labels)
  for (int k = tid; k < (p.N + 1) * K1; k += NT) ST_S(&s_binom[k], LD_G(&((const I*)p.binom)[k]));
  for (int k = tid; k < p.nb; k += NT) {
    const BondDev b = LD_G(&p.bonds[k]);
    CBond<R> sb;
    sb.mask = b.mask; sb.Jh = (R)b.Jh; sb.Jq = (R)b.Jq; sb.i = b.i; sb.j = b.j;
    ST_S(&s_bonds[k], sb);
  }
  const int chain = blockIdx.x;
  const uint64_t key = LD_G(&keys[chain]);
  int iq = 0, ip = 1, iy = 2;                               // roles of the three buffers: q_j, q_{j-1}, y
  // ---- start vector: g / ||g|| with an FP64 norm (reading 12), q_0 = 0 ---------------------------------------
  {
    double s = 0.0, z1 = 0.0, z2 = 0.0;
    for (int t = tid; t < D; t += NT) { const double g = gauss_elem(key, (uint64_t)t); s += g * g; }
    block_sum3(s, z1, z2, s_red);
    if (tid == 0) { s_sc[5] = sqrt(s); s_sc[0] = 0.0; s_sc[3] = 0.0; s_sc[4] = 0.0; }
    __syncthreads();
    const double nrm = s_sc[5];
    for (int t = tid; t < D; t += NT) {
      ST_S(&vec[(size_t)iq * vstride + t], (R)(gauss_elem(key, (uint64_t)t) / nrm));
      ST_S(&vec[(size_t)ip * vstride + t], (R)0);
    }
  }
  if (p.labels) {                                          // (s_binom was written by other threads: the barrier inside block_sum3 above orders it)
    for (int t = tid; t < D; t += NT) ST_S(&lab[t], unrank<L, I>((I)t, p.N, K1, p.K, s_binom));
  }
  __syncthreads();
  int steps = 0;
  for (int j = 0; j < p.limit; ++j) {
    const R* q = vec + (size_t)iq * vstride;
    const R* qp = vec + (size_t)ip * vstride;
    R* y = vec + (size_t)iy * vstride;
    const R bprev = (R)s_sc[0];
    double s_qy = 0.0, s_yy = 0.0, s_qq = 0.0;
    for (int t = tid; t < D; t += NT) {
      const L n = p.labels ? LD_S(&lab[t]) : unrank<L, I>((I)t, p.N, K1, p.K, s_binom);
      R acc = 0, danti = 0;
      for (int b = 0; b < p.nb; ++b) {
        const CBond<R> bd = LD_S(&s_bonds[b]);
        const L m = (L)bd.mask;
        const L x = n & m;
        if (x != 0 && x != m) {                                   // antiparallel spins
          I idx;
          if (MODE == FTLM_INDEX_CLT) idx = (I)clt_lookup((uint32_t)(n ^ m), p.clt);
          else if (MODE == FTLM_INDEX_LIN) idx = (I)lin_lookup((uint64_t)(n ^ m), p.lin_h, p.lin_hi, p.lin_lo);
          else idx = (I)t + cr_delta<L, I>(n, bd.i, bd.j, K1, s_binom);
          acc += bd.Jh * LD_S(&q[idx]);
          danti += bd.Jq;
        }
      }
      const R vt = LD_S(&q[t]);
      R out = ((R)p.diag0 - 2 * danti) * vt + acc;
      out -= bprev * LD_S(&qp[t]);
      s_qy += (double)vt * (double)out;
      s_yy += (double)out * (double)out;
      s_qq += (double)vt * (double)vt;
      ST_S(&y[t], out);
    }
    block_sum3(s_qy, s_yy, s_qq, s_red);                   // (has the barriers that order y's stores before its reads)
    if (tid == 0) {
      const double a = s_qy, b = s_yy, c = s_qq;
      const double alpha = c > 0.0 ? a / c : 0.0;
      double b2 = c > 0.0 ? b - a * a / c : 0.0;
      if (!(b2 > 0.0)) b2 = 0.0;
      const double beta = sqrt(b2);
      ST_G(&p.alpha[(size_t)chain * p.limit + j], alpha);
      ST_G(&p.beta[(size_t)chain * p.limit + j], beta);
      const double sc = fmax(s_sc[3], fmax(fabs(alpha), beta));
      s_sc[3] = sc; s_sc[1] = alpha; s_sc[2] = beta > 0.0 ? 1.0 / beta : 0.0; s_sc[0] = beta;
      s_sc[4] = (j + 1 >= p.limit || beta <= p.tol * sc) ? 1.0 : 0.0;
    }
    __syncthreads();
    steps = j + 1;
    if (s_sc[4] != 0.0) break;                              // uniform: every thread reads the same flag
    const R a = (R)s_sc[1], ib = (R)s_sc[2];
    R* qn = vec + (size_t)ip * vstride;                     // q_{j+1} over q_{j-1}
    for (int t = tid; t < D; t += NT) ST_S(&qn[t], (LD_S(&y[t]) - a * LD_S(&q[t])) * ib);
    const int old_q = iq; iq = ip; ip = old_q;              // q_{j+1} <-> q_j; y stays
    __syncthreads();
  }
  if (tid == 0) ST_G(&p.m_eff[chain], steps);
}

}  // namespace

bool ftlm_chain_persistent_fits(const ftlm_ctx* c) {
  if (c->dim < 1 || c->dim > (1 << 20)) return false;
  const int isz = c->idx64 ? 8 : 4;
  const size_t need = chain_smem_bytes(c->N, c->N_up, c->nb, c->dim, (int)ftlm_elem_size(c), isz, c->prec == FTLM_FP32 ? (int)sizeof(CBond<float>) : (int)sizeof(CBond<double>), 0);
  return need <= (size_t)227 * 1024 - 1024;
}

uint64_t ftlm_chain_key(uint64_t seed, int N_up, int r);

template <typename R, typename L, typename I>
static int launch_chain(ftlm_ctx* c, const ChainParams& p, const uint64_t* d_keys, int nchains, size_t smem, cudaStream_t s) {
#define LCH(MODE)                                                                                      \
  do {                                                                                                 \
    auto k = lanczos_chain_kernel<R, L, I, MODE>;                                                       \
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));               \
    FTLM_LAUNCH(k, nchains, CHAIN_THREADS, smem, s, p, d_keys);                                         \
  } while (0)
  if (c->mode == FTLM_INDEX_CLT) LCH(FTLM_INDEX_CLT); else if (c->mode == FTLM_INDEX_LIN) LCH(FTLM_INDEX_LIN); else LCH(FTLM_INDEX_CR);
#undef LCH
  CK(cudaGetLastError());
  return FTLM_OK;
}

int ftlm_launch_chain_persistent(ftlm_ctx* c, uint64_t seed, int r0, int nchains, int limit, double* d_alpha, double* d_beta,
                                 int* d_m_eff, cudaStream_t s) {
  if (!ftlm_chain_persistent_fits(c)) { ftlm_set_error("persistent chain kernel: the sector does not fit shared memory"); return FTLM_EUNSUPPORTED; }
  if (nchains < 1 || limit < 1) { ftlm_set_error("persistent chain kernel: bad argument"); return FTLM_EINVAL; }
  std::vector<uint64_t> keys((size_t)nchains);
  for (int r = 0; r < nchains; ++r) keys[(size_t)r] = ftlm_chain_key(seed, c->N_up, r0 + r);
  uint64_t* d_keys = nullptr;
  if (ftlm_dmalloc(&d_keys, keys.size() * 8) != cudaSuccess) { cudaGetLastError(); ftlm_set_error("persistent chain kernel: out of device memory"); return FTLM_ENOMEM; }
  int rc = FTLM_OK;
  if (cudaMemcpyAsync(d_keys, keys.data(), keys.size() * 8, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = ftlm_cuda_fail(cudaGetLastError(), "persistent chain kernel: keys");
  ChainParams p;
  p.N = c->N; p.K = c->N_up; p.nb = c->nb; p.mode = c->mode; p.limit = limit;
  p.lin_h = c->lin_h; p.lin_hi = c->d_lin_hi; p.lin_lo = c->d_lin_lo; p.dim = c->dim;
  p.binom = c->idx64 ? (const void*)c->d_binom64 : (const void*)c->d_binom32;
  p.bonds = c->d_bonds; p.clt = c->d_clt; p.diag0 = c->diag0; p.tol = c->prec == FTLM_FP32 ? 1e-5 : 1e-12;
  p.alpha = d_alpha; p.beta = d_beta; p.m_eff = d_m_eff;
  const int isz = c->idx64 ? 8 : 4, lsz = c->lab64 ? 8 : 4;
  const int esz0 = (int)ftlm_elem_size(c), bsz0 = c->prec == FTLM_FP32 ? (int)sizeof(CBond<float>) : (int)sizeof(CBond<double>);
  p.labels = chain_smem_bytes(c->N, c->N_up, c->nb, c->dim, esz0, isz, bsz0, lsz) <= (size_t)227 * 1024 - 1024 ? 1 : 0;
  const int lz = p.labels ? lsz : 0;
  if (rc == FTLM_OK) {
    if (c->prec == FTLM_FP32) {
      const size_t smem = chain_smem_bytes(c->N, c->N_up, c->nb, c->dim, 4, isz, (int)sizeof(CBond<float>), lz);
      rc = !c->lab64 ? launch_chain<float, uint32_t, uint32_t>(c, p, d_keys, nchains, smem, s)
                     : launch_chain<float, uint64_t, uint32_t>(c, p, d_keys, nchains, smem, s);
    } else {
      const size_t smem = chain_smem_bytes(c->N, c->N_up, c->nb, c->dim, 8, isz, (int)sizeof(CBond<double>), lz);
      rc = !c->lab64 ? launch_chain<double, uint32_t, uint32_t>(c, p, d_keys, nchains, smem, s)
                     : launch_chain<double, uint64_t, uint32_t>(c, p, d_keys, nchains, smem, s);
    }
  }
  if (cudaStreamSynchronize(s) != cudaSuccess && rc == FTLM_OK) rc = ftlm_cuda_fail(cudaGetLastError(), "persistent chain kernel");
  ftlm_dfree(d_keys);
  return rc;
}
