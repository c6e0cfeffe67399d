// PASS-B: index arithmetic shared by the PASS-B kernel (ftlm_passb.cu) and by the
// neighbour-index test hook of the TML kernels (ftlm_tml.cu).
//
// A window S = [lo, lo+s) of label positions is "active", the f = N - lo - s positions above are
// frozen (F) and the lo positions below are a passive batch index: for fixed hi = (F << s) | u the
// rows with every admissible low part are one contiguous run of C(lo, kP) rows,
// kP = N_up - popc(hi), ordered by the rank of the low part.  run_start(hi) is the sector index of
// the first row of that run = the index of the label (hi << lo) | (2^kP - 1):
//   CR  (Alg. 1, at d = 2): sum over the set bits p of the label of C(p, c_p); the low
//        part 2^kP - 1 contributes sum_q C(q, q+1) = 0, a set bit p of hi contributes
//        C(p + lo, kP + number of set bits of hi at or below p);
//   CLT (Alg. 2): C_b + popc(M_b & (2^j - 1)) for the block b = label >> 5, j = label & 31.
#pragma once
#include "ftlm_common.cuh"

#ifdef __CUDACC__
template <int MODE>
__device__ __forceinline__ uint64_t passb_run_start(uint64_t hi, int lo, int kP, int K,
                                                    const uint64_t* __restrict__ binom,
                                                    const uint2* __restrict__ clt) {
  if (MODE == FTLM_INDEX_CLT) {
    const uint64_t n0 = (hi << lo) | ((1ull << kP) - 1ull);
    const uint2 e = LDG(&clt[n0 >> 5]);
    const uint32_t j = (uint32_t)n0 & 31u;
    return (uint64_t)e.y + (uint64_t)__popc(e.x & ((1u << j) - 1u));
  }
  const int K1 = K + 1;
  uint64_t r = 0, x = hi;
  int c = kP;
  while (x) {
    const int p = __ffsll((long long)x) - 1;
    x &= x - 1;
    ++c;
    r += LD_A(&binom[(p + lo) * K1 + c]);
  }
  return r;
}

// Rank of the low part (lo bits, popcount kP) inside its run: sum over set bits q of C(q, ordinal).
__device__ __forceinline__ uint64_t passb_low_rank(uint64_t low, int K, const uint64_t* __restrict__ binom) {
  const int K1 = K + 1;
  uint64_t r = 0;
  int c = 0;
  while (low) {
    const int q = __ffsll((long long)low) - 1;
    low &= low - 1;
    ++c;
    r += LD_A(&binom[q * K1 + c]);
  }
  return r;
}
#endif  // __CUDACC__
