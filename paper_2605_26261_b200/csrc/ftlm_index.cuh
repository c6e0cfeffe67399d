// Index arithmetic shared by the thread-per-row kernels (ftlm_row.cu) and the persistent chain kernel
// (ftlm_chain.cu): inverse map (L136), Algorithm 1 (L138-L144) and its incremental form, Algorithm 2
// (L167-L173), Lin's two tables (L119).  Internal.
#pragma once
#include "ftlm_common.cuh"

#ifdef __CUDACC__
namespace {

// Inverse map (L136; reading 26): at bit p with A ones left, bit p = 1 iff r >= C(p, A).
// binom is the (saturated) table [p*(K+1) + a] in shared memory.
template <typename L, typename I>
__device__ __forceinline__ L unrank(I r, int N, int K1, int K, const I* __restrict__ binom) {
  L n = 0;
  int A = K;
  for (int p = N - 1; p >= 0 && A > 0; --p) {
    const I c = LD_S(&binom[p * K1 + A]);
    if (r >= c) { n |= (L)1 << p; r -= c; --A; }
  }
  return n;
}

// Algorithm 1 (L138-L144) at d = 2: rank += D_c(p, A, a_p) = a_p ? C(p, A) : 0; A -= a_p.
template <typename L, typename I>
__device__ __forceinline__ I rank_alg1(L x, int N, int K1, int K, const I* __restrict__ binom) {
  I rank = 0;
  int A = K;
  for (int p = N - 1; p >= 0; --p) {
    if ((x >> p) & 1) { rank += LD_S(&binom[p * K1 + A]); --A; }
  }
  return rank;
}

// Incremental CR: index change when the one of an antiparallel bond (i < j) moves.
// Only the binomial terms of positions i..j change.  Unsigned wrap-around is harmless.
template <typename L, typename I>
__device__ __forceinline__ I cr_delta(L x, int i, int j, int K1, const I* __restrict__ binom) {
  const int ci = popc_((L)(x & ((((L)2) << i) - 1)));         // ones at positions <= i
  const int cj = popc_((L)(x & ((((L)2) << j) - 1)));         // ones at positions <= j
  L between = x & ((((L)1) << j) - 1) & ~((((L)2) << i) - 1);
  I d;
  int c = ci;
  if ((x >> j) & 1) {                                          // the one moves down j -> i
    d = LD_S(&binom[i * K1 + ci + 1]) - LD_S(&binom[j * K1 + cj]);
    while (between) {
      const int p = ffs_(between) - 1;
      between &= between - 1;
      ++c;
      d += LD_S(&binom[p * K1 + c + 1]) - LD_S(&binom[p * K1 + c]);
    }
  } else {                                                     // the one moves up i -> j
    d = LD_S(&binom[j * K1 + cj]) - LD_S(&binom[i * K1 + ci]);
    while (between) {
      const int p = ffs_(between) - 1;
      between &= between - 1;
      ++c;
      d += LD_S(&binom[p * K1 + c - 1]) - LD_S(&binom[p * K1 + c]);
    }
  }
  return d;
}

// Algorithm 2 (L167-L173): b = n >> 5, j = n & 31, index = C_b + popc(M_b & (2^j - 1)).
__device__ __forceinline__ int64_t clt_lookup_checked(uint64_t n, int N, const uint2* __restrict__ clt) {
  if (N < 64 && (n >> N)) return -1;
  const uint2 e = LD_G(&clt[n >> 5]);
  const uint32_t j = (uint32_t)n & 31u;
  if (!((e.x >> j) & 1u)) return -1;
  return (int64_t)e.y + __popc(e.x & ((1u << j) - 1u));
}
__device__ __forceinline__ uint32_t clt_lookup(uint32_t n, const uint2* __restrict__ clt) {
  const uint2 e = LDG(&clt[n >> 5]);
  return e.y + __popc(e.x & ((1u << (n & 31u)) - 1u));
}

// Lin's two-table lookup (L119): index = Ja[n >> h] + Jb[n & (2^h - 1)] for an in-sector label n.
__device__ __forceinline__ uint64_t lin_lookup(uint64_t n, int h, const uint64_t* __restrict__ Ja, const uint32_t* __restrict__ Jb) {
  return LDG(&Ja[n >> h]) + (uint64_t)LDG(&Jb[n & ((1ull << h) - 1ull)]);
}

}  // namespace
#endif  // __CUDACC__
