// Memory-access wrappers of libftlm's kernels (internal; included by ftlm_common.cuh).
//
// Every load, store, asynchronous copy and atomic a kernel makes through a COMPUTED address goes
// through one of the macros below.  Three builds of the same kernel sources:
//   release       each macro is the bare access (identical code to writing it out);
//   FTLM_CHECKED  the address is tested first - natural alignment, and membership in the table of
//                 live device ranges (library allocations + the caller buffers of recent calls) for
//                 global memory, or in the CTA's dynamic shared-memory window for shared memory.
//                 A violation SUPPRESSES the access (loads give zero), bumps a device counter and
//                 records the first (translation unit, source line, address, block, thread).
//                 It never traps: a trap is itself an Xid on the device.  The library reports the
//                 count through ftlm_get_option(ctx, "check_violations"); tests/conftest.py runs the
//                 GPU suite in this build first and refuses the release build unless it is zero.
//   FTLM_EMU      (host emulation, tests/emu) natural alignment is asserted - x86 tolerates the
//                 misaligned vector accesses that raise Xid 13 on the device - and ranges are the
//                 emulation's guard pages.
#pragma once
#include <stdint.h>

#define FTLM_CHK_MAX_RANGES 512
#define FTLM_CHK_CALL_RANGES 16

struct FtlmChkRange { unsigned long long lo, hi; };   // [lo, hi)
struct FtlmChkState {
  unsigned long long violations;
  unsigned long long first_addr;
  int first_tu, first_line, first_block, first_thread, first_kind, first_bytes;   // kind: 0 global range, 1 global alignment, 2 shared range, 3 shared alignment
  int n_ranges, pad;
  FtlmChkRange call[FTLM_CHK_CALL_RANGES];          // caller buffers of recent API calls (unsorted; hi == 0: empty)
  FtlmChkRange ranges[FTLM_CHK_MAX_RANGES];          // library allocations, sorted by lo, disjoint
};

#ifndef FTLM_TU
#define FTLM_TU 0
#endif

#if defined(FTLM_CHECKED) && !defined(FTLM_EMU)
// ---------------------------------------------------------------------------------------------
static __device__ FtlmChkState* ftlm_chk_dev;        // one copy per translation unit, bound before its first launch

__device__ __noinline__ static bool ftlm_chk_fail(unsigned long long addr, int bytes, int line, int kind) {
  FtlmChkState* s = ftlm_chk_dev;
  if (s && atomicAdd(&s->violations, 1ull) == 0ull) {
    s->first_addr = addr; s->first_tu = FTLM_TU; s->first_line = line; s->first_block = (int)blockIdx.x;
    s->first_thread = (int)threadIdx.x; s->first_kind = kind; s->first_bytes = bytes;
  }
  return false;
}

__device__ __noinline__ static bool ftlm_chk_g(const void* p, int bytes, int align, int line) {
  const FtlmChkState* s = ftlm_chk_dev;
  const unsigned long long a = (unsigned long long)p;
  if (!s) return true;                                 // not bound: cannot happen after ftlm_chk_bind_tu()
  if (a & (unsigned long long)(align - 1)) return ftlm_chk_fail(a, bytes, line, 1);
#pragma unroll 1
  for (int k = 0; k < FTLM_CHK_CALL_RANGES; ++k)
    if (a >= s->call[k].lo && a + (unsigned long long)bytes <= s->call[k].hi) return true;
  int lo = 0, hi = s->n_ranges;                        // last range with ranges[k].lo <= a
#pragma unroll 1
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (s->ranges[mid].lo <= a) lo = mid + 1; else hi = mid;
  }
  if (lo > 0 && a + (unsigned long long)bytes <= s->ranges[lo - 1].hi) return true;
  return ftlm_chk_fail(a, bytes, line, 0);
}

__device__ __noinline__ static bool ftlm_chk_s(const void* p, int bytes, int align, int line) {
  extern __shared__ __align__(16) unsigned char ftlm_chk_dyn_[];   // every extern array starts at the dynamic shared-memory base
  unsigned dyn;
  asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
  const unsigned long long a = (unsigned long long)p;
  if (a & (unsigned long long)(align - 1)) return ftlm_chk_fail(a, bytes, line, 3);
  if (!__isShared(p)) return ftlm_chk_fail(a, bytes, line, 2);
  const unsigned sa = (unsigned)__cvta_generic_to_shared(p), sb = (unsigned)__cvta_generic_to_shared(ftlm_chk_dyn_);
  if (sa < sb || sa + (unsigned)bytes > sb + dyn) return ftlm_chk_fail(a, bytes, line, 2);
  return true;
}
#define FTLM_G_OK(p, T, line) ftlm_chk_g((const void*)(p), (int)sizeof(T), (int)alignof(T), (line))
#define FTLM_S_OK(p, T, line) ftlm_chk_s((const void*)(p), (int)sizeof(T), (int)alignof(T), (line))
#define FTLM_G_OKN(p, bytes, align, line) ftlm_chk_g((const void*)(p), (int)(bytes), (int)(align), (line))   /* a whole range (bulk copy) */
#define FTLM_S_OKN(p, bytes, align, line) ftlm_chk_s((const void*)(p), (int)(bytes), (int)(align), (line))
#define FTLM_A_OK(p, T, line) (__isShared((const void*)(p)) ? FTLM_S_OK(p, T, line) : FTLM_G_OK(p, T, line))

#elif defined(FTLM_EMU)
// ---------------------------------------------------------------------------------------------
static inline bool ftlm_emu_aligned(const void* p, size_t align, int line, const char* what) {
  if (((uintptr_t)p & (align - 1)) != 0) {
    fprintf(stderr, "cuda_emu: misaligned %s of %zu-byte-aligned type at %p (tu %d line %d, block %u thread %u)\n", what, align, p,
            FTLM_TU, line, blockIdx.x, threadIdx.x);
    fflush(stderr);
    abort();
  }
  return true;
}
// shared-memory accesses also feed the emulation's race detector (cuda_emu::smem_access: per-word last writer /
// reader and the barrier epochs they were made in; two accesses of different threads to one word, one of them a
// write, with no __syncthreads / __syncwarp between them abort the run)
#define FTLM_G_OK(p, T, line) ftlm_emu_aligned((const void*)(p), alignof(T), (line), "global access")
#define FTLM_S_OK(p, T, line) (ftlm_emu_aligned((const void*)(p), alignof(T), (line), "shared access") && cuda_emu::smem_access((const void*)(p), sizeof(T), false, FTLM_TU, (line)))
#define FTLM_SW_OK(p, T, line) (ftlm_emu_aligned((const void*)(p), alignof(T), (line), "shared access") && cuda_emu::smem_access((const void*)(p), sizeof(T), true, FTLM_TU, (line)))
#define FTLM_A_OK(p, T, line) (ftlm_emu_aligned((const void*)(p), alignof(T), (line), "access") && cuda_emu::smem_access((const void*)(p), sizeof(T), false, FTLM_TU, (line)))
#define FTLM_G_OKN(p, bytes, align, line) ftlm_emu_aligned((const void*)(p), (align), (line), "bulk-copy source")
#define FTLM_S_OKN(p, bytes, align, line) ftlm_emu_aligned((const void*)(p), (align), (line), "bulk-copy destination")

#else
#define FTLM_G_OK(p, T, line) true
#define FTLM_S_OK(p, T, line) true
#define FTLM_A_OK(p, T, line) true
#define FTLM_G_OKN(p, bytes, align, line) true
#define FTLM_S_OKN(p, bytes, align, line) true
#endif
#ifndef FTLM_SW_OK
#define FTLM_SW_OK(p, T, line) FTLM_S_OK(p, T, line)      /* shared-memory WRITE (the emulation's race detector tells them apart) */
#endif

#ifdef __CUDACC__
namespace fa {
template <typename T> __device__ __forceinline__ T ld_g(const T* p, int line) { if (!FTLM_G_OK(p, T, line)) return T{}; return *p; }
template <typename T> __device__ __forceinline__ T ldg(const T* p, int line) { if (!FTLM_G_OK(p, T, line)) return T{}; return __ldg(p); }
template <typename T> __device__ __forceinline__ T ldcs(const T* p, int line) { if (!FTLM_G_OK(p, T, line)) return T{}; return __ldcs(p); }
template <typename T, typename U> __device__ __forceinline__ void st_g(T* p, const U& v, int line) { if (FTLM_G_OK(p, T, line)) *p = (T)v; }
template <typename T, typename U> __device__ __forceinline__ void stcs(T* p, const U& v, int line) { if (FTLM_G_OK(p, T, line)) __stcs(p, (T)v); }
template <typename T> __device__ __forceinline__ T ld_s(const T* p, int line) { if (!FTLM_S_OK(p, T, line)) return T{}; return *p; }
// predicated shared-memory load: `other` for lanes whose condition is false.  (In the emulation every lane passes
// here, which keeps the per-thread occurrence numbers of the shared-memory profile aligned across the lanes of a warp.)
template <typename T> __device__ __forceinline__ T ld_s_if(bool c, const T* p, const T& other, int line) {
#ifdef FTLM_EMU
  if (!c) { cuda_emu::smem_skip(FTLM_TU, line); return other; }
#else
  if (!c) return other;
#endif
  if (!FTLM_S_OK(p, T, line)) return T{};
  return *p;
}
template <typename T, typename U> __device__ __forceinline__ void st_s(T* p, const U& v, int line) { if (FTLM_SW_OK(p, T, line)) *p = (T)v; }
template <typename T> __device__ __forceinline__ T ld_a(const T* p, int line) { if (!FTLM_A_OK(p, T, line)) return T{}; return *p; }
template <typename T> __device__ __forceinline__ T atom_add_g(T* p, T v, int line) { if (!FTLM_G_OK(p, T, line)) return T{}; return atomicAdd(p, v); }
}  // namespace fa

#define LD_G(p) fa::ld_g((p), __LINE__)          /* plain global load */
#define LDG(p) fa::ldg((p), __LINE__)            /* read-only (non-coherent) global load */
#define LDCS(p) fa::ldcs((p), __LINE__)          /* streaming global load */
#define ST_G(p, ...) fa::st_g((p), (__VA_ARGS__), __LINE__)  /* plain global store */
#define STCS(p, ...) fa::stcs((p), (__VA_ARGS__), __LINE__)  /* streaming global store */
#define LD_S(p) fa::ld_s((p), __LINE__)          /* shared-memory load */
#define LD_S_IF(c, p, other) fa::ld_s_if((c), (p), (other), __LINE__)   /* predicated shared-memory load */
#define ST_S(p, ...) fa::st_s((p), (__VA_ARGS__), __LINE__)  /* shared-memory store */
#define LD_A(p) fa::ld_a((p), __LINE__)          /* load through a pointer that is shared in some callers, global in others */
#define ATOM_ADD_G(p, ...) fa::atom_add_g((p), (__VA_ARGS__), __LINE__)
#endif  // __CUDACC__
