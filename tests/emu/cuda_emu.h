// cuda_emu.h - TEST INFRASTRUCTURE: a minimal SIMT emulation of the CUDA constructs that libftlm's
// kernels use, so that the SAME kernel sources (paper_2605_26261_b200/csrc/*.cu, compiled as C++
// with -DFTLM_EMU) can be executed on the host by `-m "not gpu"` tests: every CUDA thread of a CTA is
// a fiber (ucontext), __syncthreads / __syncwarp / __ballot_sync / __shfl_*_sync are real rendezvous
// points, "device" memory is guarded host memory (a PROT_NONE page directly behind every allocation
// and behind the dynamic shared memory, so reads or writes past the end fault instead of passing).
// The CTAs of a grid run CONCURRENTLY on a few host threads (FTLM_EMU_CTAS, default 4; each CTA's fibers stay on one
// host thread), taken from a shared counter like a hardware scheduler would: the atomic tile / item hand-out, the
// last-CTA ticket and the counter reset of the persistent kernels really race; atomics are real atomics.
// Shared-memory race detector: every access made through the LD_S / ST_S / cp_async macros of csrc/ftlm_access.cuh
// is recorded per 4-byte word (last writer, last reader, the __syncthreads / __syncwarp epochs they were made in);
// two accesses to one word by different threads, at least one a write, with no barrier between them abort the run
// (FTLM_EMU_RACE=0 turns the detector off).
// FTLM_EMU_ALIGN=front places every allocation flush against its FRONT guard page instead of the back one, so
// that underruns fault too (the suite is run both ways).  This is a checker for index arithmetic, table construction,
// barrier placement, cp.async waits, alignment and bounds - it is never loaded by the product binding and has no performance
// meaning.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>

#define __host__
#define __device__
#define __global__
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __grid_constant__
#define __align__(n) __attribute__((aligned(n)))
#define __shared__ static thread_local      // one copy per host thread = per CTA in flight
#ifndef __CUDACC__
#define __CUDACC__ 1          // ftlm_common.cuh guards its device helpers with this
#endif

struct uint3 { unsigned x, y, z; };
struct dim3 { unsigned x = 1, y = 1, z = 1; dim3() {} dim3(unsigned a, unsigned b = 1, unsigned c = 1) : x(a), y(b), z(c) {} };
struct __attribute__((aligned(8))) float2 { float x, y; };
struct __attribute__((aligned(16))) float4 { float x, y, z, w; };
struct __attribute__((aligned(16))) double2 { double x, y; };
struct __attribute__((aligned(8))) uint2 { unsigned x, y; };
struct __attribute__((aligned(16))) uint4 { unsigned x, y, z, w; };
struct __attribute__((aligned(8))) int2 { int x, y; };
static inline uint2 make_uint2(unsigned a, unsigned b) { return uint2{a, b}; }
static inline uint4 make_uint4(unsigned a, unsigned b, unsigned c, unsigned d) { return uint4{a, b, c, d}; }
static inline float2 make_float2(float a, float b) { return float2{a, b}; }
static inline float4 make_float4(float a, float b, float c, float d) { return float4{a, b, c, d}; }
static inline double2 make_double2(double a, double b) { return double2{a, b}; }
static inline int2 make_int2(int a, int b) { return int2{a, b}; }

extern thread_local uint3 threadIdx, blockIdx;
extern thread_local dim3 blockDim, gridDim;

// ---- runtime API subset ------------------------------------------------------------------------
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2, cudaErrorNoDevice = 100 };
typedef struct cuda_emu_stream* cudaStream_t;
typedef struct cuda_emu_event* cudaEvent_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost = 0, cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
struct cudaDeviceProp { char name[256]; int multiProcessorCount; size_t sharedMemPerBlockOptin; int major, minor; size_t l2CacheSize; };

cudaError_t cudaGetDeviceCount(int* n);
cudaError_t cudaSetDevice(int d);
cudaError_t cudaGetDeviceProperties(cudaDeviceProp* p, int d);
cudaError_t cudaMalloc(void** p, size_t bytes);
template <typename T> static inline cudaError_t cudaMalloc(T** p, size_t bytes) { return cudaMalloc((void**)p, bytes); }
cudaError_t cudaFree(void* p);
cudaError_t cudaMemcpy(void* dst, const void* src, size_t bytes, cudaMemcpyKind k);
cudaError_t cudaMemcpyAsync(void* dst, const void* src, size_t bytes, cudaMemcpyKind k, cudaStream_t s = nullptr);
cudaError_t cudaMemset(void* p, int v, size_t bytes);
cudaError_t cudaMemsetAsync(void* p, int v, size_t bytes, cudaStream_t s = nullptr);
cudaError_t cudaGetLastError();
cudaError_t cudaPeekAtLastError();
const char* cudaGetErrorString(cudaError_t e);
cudaError_t cudaDeviceSynchronize();
cudaError_t cudaStreamSynchronize(cudaStream_t s);
cudaError_t cudaEventCreate(cudaEvent_t* e);
cudaError_t cudaEventDestroy(cudaEvent_t e);
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t s = nullptr);
cudaError_t cudaEventSynchronize(cudaEvent_t e);
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b);
template <typename F> static inline cudaError_t cudaFuncSetAttribute(F, cudaFuncAttribute, int) { return cudaSuccess; }
template <typename F> static inline cudaError_t cudaOccupancyMaxActiveBlocksPerMultiprocessor(int* n, F, int threads, size_t smem) {
  size_t by_smem = smem ? (size_t)(227 * 1024) / (smem + 1024) : 32;
  int by_thr = 2048 / (threads > 0 ? threads : 1);
  *n = (int)std::min<size_t>(by_smem, (size_t)by_thr);
  return cudaSuccess;
}

// ---- launch ------------------------------------------------------------------------------------
namespace cuda_emu {
void launch(unsigned grid, unsigned block, size_t dyn_smem, const std::function<void()>& body);
unsigned char* dyn_smem();
void sync_threads();
uint64_t collective(int op, unsigned mask, uint64_t v, int arg);
// cp.async model: the destination is poisoned (0xFF bytes = NaN) when the copy is issued and the bytes land
// only when the ISSUING thread executes cp_async_wait_all(); a thread that exits with copies pending aborts.
// A consumer that reads before the producer's wait + barrier therefore sees NaN instead of passing by luck.
void cp_async_issue(void* smem_dst, const void* gsrc, size_t bytes);
void cp_async_wait_all();
// Bulk copy + mbarrier model (cp.async.bulk ... mbarrier::complete_tx::bytes): the destination is poisoned when the
// copy is issued (and the issue counts as a write of the issuing thread for the race detector: readers of the old
// content must have passed a barrier); the bytes land when some thread's mbar_wait finds all arrivals made and then
// completes the phase.  Size, source and destination must be multiples of 16 bytes.
void mbar_init(void* mbar, int count);
void mbar_arrive_expect_tx(void* mbar, unsigned bytes);
void bulk_issue(void* smem_dst, const void* gsrc, unsigned bytes, void* mbar, int tu, int line);
void mbar_wait(void* mbar, unsigned parity);
// race detector hook (always returns true); a pointer outside the CTA's dynamic shared memory is ignored
bool smem_access(const void* p, size_t bytes, bool write, int tu, int line);
// profile only: an inactive lane of a predicated shared-memory load passes the instruction (occurrence numbering)
void smem_skip(int tu, int line);
enum { OP_SYNCWARP = 0, OP_BALLOT = 1, OP_SHFL_DOWN = 2, OP_SHFL_XOR = 3, OP_SHFL_IDX = 4, OP_SHFL_UP = 5 };
template <typename T> static inline uint64_t pack(T v) { uint64_t u = 0; static_assert(sizeof(T) <= 8, "shfl payload"); memcpy(&u, &v, sizeof(T)); return u; }
template <typename T> static inline T unpack(uint64_t u) { T v; memcpy(&v, &u, sizeof(T)); return v; }
}  // namespace cuda_emu

#define FTLM_LAUNCH(kernel, grid, block, smem, stream, ...) \
  cuda_emu::launch((unsigned)(grid), (unsigned)(block), (size_t)(smem), [&]() { kernel(__VA_ARGS__); })
#define FTLM_DYN_SMEM(name) unsigned char* name = cuda_emu::dyn_smem()

// ---- intrinsics --------------------------------------------------------------------------------
static inline void __syncthreads() { cuda_emu::sync_threads(); }
static inline void __syncwarp(unsigned mask = 0xffffffffu) { cuda_emu::collective(cuda_emu::OP_SYNCWARP, mask, 0, 0); }
static inline unsigned __ballot_sync(unsigned mask, int pred) { return (unsigned)cuda_emu::collective(cuda_emu::OP_BALLOT, mask, pred ? 1 : 0, 0); }
template <typename T> static inline T __shfl_down_sync(unsigned mask, T v, int d) { return cuda_emu::unpack<T>(cuda_emu::collective(cuda_emu::OP_SHFL_DOWN, mask, cuda_emu::pack(v), d)); }
template <typename T> static inline T __shfl_up_sync(unsigned mask, T v, int d) { return cuda_emu::unpack<T>(cuda_emu::collective(cuda_emu::OP_SHFL_UP, mask, cuda_emu::pack(v), d)); }
template <typename T> static inline T __shfl_xor_sync(unsigned mask, T v, int d) { return cuda_emu::unpack<T>(cuda_emu::collective(cuda_emu::OP_SHFL_XOR, mask, cuda_emu::pack(v), d)); }
template <typename T> static inline T __shfl_sync(unsigned mask, T v, int src) { return cuda_emu::unpack<T>(cuda_emu::collective(cuda_emu::OP_SHFL_IDX, mask, cuda_emu::pack(v), src)); }
static inline void __threadfence() { __atomic_thread_fence(__ATOMIC_SEQ_CST); }
static inline void __threadfence_block() { __atomic_thread_fence(__ATOMIC_SEQ_CST); }
static inline int __popc(unsigned x) { return __builtin_popcount(x); }
static inline int __popcll(unsigned long long x) { return __builtin_popcountll(x); }
static inline int __ffs(int x) { return __builtin_ffs(x); }
static inline int __ffsll(long long x) { return __builtin_ffsll(x); }
static inline int __clz(int x) { return x ? __builtin_clz((unsigned)x) : 32; }
static inline float __uint_as_float(unsigned u) { float f; memcpy(&f, &u, 4); return f; }
static inline unsigned __float_as_uint(float f) { unsigned u; memcpy(&u, &f, 4); return u; }
template <typename T> static inline T __ldg(const T* p) { return *p; }
template <typename T> static inline T __ldcs(const T* p) { return *p; }
template <typename T> static inline T __ldcg(const T* p) { return *p; }
template <typename T> static inline void __stcs(T* p, const T& v) { *p = v; }
template <typename T> static inline void __stcg(T* p, const T& v) { *p = v; }
static inline unsigned atomicAdd(unsigned* p, unsigned v) { return __atomic_fetch_add(p, v, __ATOMIC_SEQ_CST); }
static inline int atomicAdd(int* p, int v) { return __atomic_fetch_add(p, v, __ATOMIC_SEQ_CST); }
static inline unsigned long long atomicAdd(unsigned long long* p, unsigned long long v) { return __atomic_fetch_add(p, v, __ATOMIC_SEQ_CST); }
static inline unsigned long long atomicMax(unsigned long long* p, unsigned long long v) {
  unsigned long long o = __atomic_load_n(p, __ATOMIC_SEQ_CST);
  while (o < v && !__atomic_compare_exchange_n(p, &o, v, false, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST)) {}
  return o;
}
static inline long long __double_as_longlong(double d) { long long u; memcpy(&u, &d, 8); return u; }
static inline double atomicAdd(double* p, double v) {
  uint64_t o, n;
  __atomic_load((uint64_t*)p, &o, __ATOMIC_SEQ_CST);
  for (;;) { double d; memcpy(&d, &o, 8); d += v; memcpy(&n, &d, 8); if (__atomic_compare_exchange((uint64_t*)p, &o, &n, false, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST)) { memcpy(&d, &o, 8); return d; } }
}
static inline float atomicAdd(float* p, float v) {
  uint32_t o, n;
  __atomic_load((uint32_t*)p, &o, __ATOMIC_SEQ_CST);
  for (;;) { float d; memcpy(&d, &o, 4); d += v; memcpy(&n, &d, 4); if (__atomic_compare_exchange((uint32_t*)p, &o, &n, false, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST)) { memcpy(&d, &o, 4); return d; } }
}
