// B interleaved values of R (one row of a batch of chains, L207) and their global-memory accesses (internal).
#pragma once
#include "ftlm_common.cuh"

#ifdef __CUDACC__
template <typename R, int B>
struct __align__((sizeof(R) * B) > 16 ? 16 : (sizeof(R) * B)) Vec { R x[B]; };

template <typename V> __device__ __forceinline__ V vec_ldg_(const V* p, int line) {
  V r;
  if (!FTLM_G_OK(p, V, line)) return V{};
  if constexpr (sizeof(V) == 4) *(float*)&r = __ldg((const float*)p);
  else if constexpr (sizeof(V) == 8) *(float2*)&r = __ldg((const float2*)p);
  else {
#pragma unroll
    for (int k = 0; k < (int)(sizeof(V) / 16); ++k) ((float4*)&r)[k] = __ldg((const float4*)p + k);
  }
  return r;
}
template <typename V> __device__ __forceinline__ V vec_ldcs_(const V* p, int line) {
  V r;
  if (!FTLM_G_OK(p, V, line)) return V{};
  if constexpr (sizeof(V) == 4) *(float*)&r = __ldcs((const float*)p);
  else if constexpr (sizeof(V) == 8) *(float2*)&r = __ldcs((const float2*)p);
  else {
#pragma unroll
    for (int k = 0; k < (int)(sizeof(V) / 16); ++k) ((float4*)&r)[k] = __ldcs((const float4*)p + k);
  }
  return r;
}
template <typename V> __device__ __forceinline__ void vec_stcs_(V* p, const V& r, int line) {
  if (!FTLM_G_OK(p, V, line)) return;
  if constexpr (sizeof(V) == 4) __stcs((float*)p, *(const float*)&r);
  else if constexpr (sizeof(V) == 8) __stcs((float2*)p, *(const float2*)&r);
  else {
#pragma unroll
    for (int k = 0; k < (int)(sizeof(V) / 16); ++k) __stcs((float4*)p + k, ((const float4*)&r)[k]);
  }
}
#define vec_ldg(p) vec_ldg_((p), __LINE__)
#define vec_ldcs(p) vec_ldcs_((p), __LINE__)
#define vec_stcs(p, r) vec_stcs_((p), (r), __LINE__)

// asynchronous global -> shared copy of one row of the batch (cp.async moves at most 16 bytes)
template <typename V> __device__ __forceinline__ void cp_async_vec_(V* smem_dst, const V* gsrc, int line) {
  if constexpr (sizeof(V) <= 16) cp_async_elem_(smem_dst, gsrc, line);
  else {
#pragma unroll
    for (int k = 0; k < (int)(sizeof(V) / 16); ++k) cp_async_elem_((uint4*)smem_dst + k, (const uint4*)gsrc + k, line);
  }
}
#define cp_async_vec(dst, src) cp_async_vec_((dst), (src), __LINE__)

// Last-CTA finish of a multi-pass kernel for B chains: partials[q * n + k], q = 3 b + {0: <q,y>, 1: <y,y>, 2: <q,q>},
// are added over k in a fixed assignment and order (bit-reproducible), then chain b advances (alpha_j = <q,y>/<q,q>,
// beta_j^2 = <y,y> - <q,y>^2/<q,q>, breakdown rule of reading 10).  Called by every thread of the last CTA;
// red: >= 64 + 3 B doubles of shared memory.
template <int B>
__device__ __forceinline__ void finish_chains(const double* partials, uint32_t n, ChainState* st, double* red) {
  const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
  for (int q = 0; q < 3 * B; ++q) {
    double a = 0.0;
    for (uint32_t k = tid; k < n; k += NT) a += LD_G(&partials[(size_t)q * n + k]);
    a = warp_sum(a);
    __syncthreads();
    if (lane == 0) ST_S(&red[warp], a);
    __syncthreads();
    if (tid == 0) {
      double s = 0.0;
      for (int wv = 0; wv < NW; ++wv) s += LD_S(&red[wv]);
      ST_S(&red[64 + q], s);
    }
  }
  __syncthreads();
  if (tid < B) {
    ChainState* c = st + tid;
    if (!c->done) {
      const double a = LD_S(&red[64 + 3 * tid]), b = LD_S(&red[64 + 3 * tid + 1]), cc = LD_S(&red[64 + 3 * tid + 2]);
      const int j = c->step;
      const double alpha = cc > 0.0 ? a / cc : 0.0;
      double b2 = cc > 0.0 ? b - a * a / cc : 0.0;
      if (!(b2 > 0.0)) b2 = 0.0;
      const double beta = sqrt(b2);
      c->alpha[j] = alpha;
      c->beta[j] = beta;
      double sc = c->scale;
      sc = fmax(sc, fmax(fabs(alpha), beta));
      c->scale = sc;
      c->step = j + 1;
      c->a = alpha;
      c->inv_b = beta > 0.0 ? 1.0 / beta : 0.0;
      c->beta_prev = beta;
      if (j + 1 >= c->limit || beta <= c->tol * sc) { c->done = 1; c->inv_b = 0.0; }
    }
  }
}
#endif  // __CUDACC__
