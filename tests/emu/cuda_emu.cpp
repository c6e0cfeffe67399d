// cuda_emu.cpp - TEST INFRASTRUCTURE: fiber scheduler and guarded "device" memory behind cuda_emu.h.
#include "cuda_emu.h"

#include <cstdlib>
#include <sys/mman.h>
#include <time.h>
#include <ucontext.h>
#include <unistd.h>

#include <algorithm>
#include <atomic>
#include <map>
#include <mutex>
#include <thread>
#include <vector>

thread_local uint3 threadIdx, blockIdx;
thread_local dim3 blockDim, gridDim;

namespace {

[[noreturn]] void die(const char* msg) {
  fprintf(stderr, "cuda_emu: %s (block %u thread %u)\n", msg, blockIdx.x, threadIdx.x);
  fflush(stderr);
  abort();
}

// ---- guarded allocations: [PROT_NONE page][slack ... data (16-byte aligned, ends at page end)][PROT_NONE page]
struct Alloc { void* map; size_t map_bytes; };
std::map<void*, Alloc> g_allocs;
std::mutex g_alloc_mu;
const size_t PAGE = 4096;

void* guarded_alloc(size_t bytes) {
  const size_t data = (bytes + 15) & ~(size_t)15;
  const size_t body = ((data + PAGE - 1) / PAGE) * PAGE;
  const size_t total = body + 2 * PAGE;
  char* m = (char*)mmap(nullptr, total, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0);
  if (m == MAP_FAILED) return nullptr;
  mprotect(m, PAGE, PROT_NONE);
  mprotect(m + PAGE + body, PAGE, PROT_NONE);
  static const bool front = getenv("FTLM_EMU_ALIGN") && !strcmp(getenv("FTLM_EMU_ALIGN"), "front");
  char* p = front ? m + PAGE : m + PAGE + body - data;   // data flush against the trailing (default) or the leading guard page
  memset(m + PAGE, 0xCD, body);             // slack: poison
  memset(p, 0xA5, data);                    // uninitialised device memory is not zero
  std::lock_guard<std::mutex> lk(g_alloc_mu);
  g_allocs[p] = Alloc{m, total};
  return p;
}
void guarded_free(void* p) {
  std::lock_guard<std::mutex> lk(g_alloc_mu);
  auto it = g_allocs.find(p);
  if (it == g_allocs.end()) die("cudaFree of an unknown pointer");
  munmap(it->second.map, it->second.map_bytes);
  g_allocs.erase(it);
}

// ---- fibers ------------------------------------------------------------------------------------
struct PendingCopy { void* dst; size_t bytes; unsigned char data[16]; };
struct Fiber { ucontext_t ctx; char* stack = nullptr; bool done = false; bool started = false; std::vector<PendingCopy> pending; };
struct PendingBulk { void* dst; std::vector<unsigned char> data; void* mbar; };
struct MBar { int count = 0, pending = 0; long tx = 0; unsigned completed = 0; };
thread_local std::vector<PendingBulk> g_bulk;           // bulk copies in flight of the CTA on this host thread
thread_local std::map<void*, MBar> g_mbar;
// Shared-memory profile (FTLM_EMU_PROFILE=<file>): every LD_S / ST_S / cp.async access is logged per CTA with its
// warp, lane, source line and the per-thread occurrence number of that line; at the end of the CTA the lanes of one
// warp instruction are put together and its shared-memory wavefronts are counted as on the hardware: 4-byte words
// of one instruction that fall into the same bank (word mod 32) but differ need one wavefront each.
struct ProfEv { uint32_t warp_lane; uint32_t tuline; uint32_t occ; uint32_t word; uint8_t nwords, write; };
struct ProfAgg { unsigned long long instr = 0, wavefronts = 0, ideal = 0, lanes = 0; };
thread_local std::vector<ProfEv> g_prof_ev;
thread_local std::vector<std::map<uint32_t, uint32_t>> g_prof_occ;      // per thread: occurrences of each source line
std::map<uint32_t, ProfAgg> g_prof;                                      // (tu << 20 | line) << 1 | write
std::mutex g_prof_mu;
const char* prof_path() { static const char* p = getenv("FTLM_EMU_PROFILE"); return (p && *p) ? p : nullptr; }
const size_t STACK = 64 * 1024;
// scheduler state of the CTA in flight on this host thread
thread_local std::vector<Fiber> g_fib;
thread_local std::vector<char*> g_stack_pool;
std::vector<std::vector<char*>> g_free_stack_sets;       // fiber stacks outlive the short-lived host threads of a launch
std::mutex g_stack_mu;
thread_local ucontext_t g_main;
thread_local int g_cur = -1;
thread_local unsigned g_nthreads = 0;
thread_local unsigned long long g_progress = 0;
thread_local const std::function<void()>* g_body = nullptr;
thread_local unsigned char* g_dyn = nullptr;
thread_local size_t g_dyn_bytes = 0;

// CTA barrier
thread_local unsigned g_bar_arrived = 0, g_bar_gen = 0, g_alive = 0;

// race detector: per 4-byte word of the dynamic shared memory, the last write and the last read
struct Access { int tid; unsigned bar, wgen; int tu, line; };
struct Shadow { Access w, r; };
thread_local std::vector<Shadow> g_shadow;
bool race_on() { static const bool on = !(getenv("FTLM_EMU_RACE") && !strcmp(getenv("FTLM_EMU_RACE"), "0")); return on; }

struct Warp {
  uint64_t val[32], out[32];
  int arg[32];
  unsigned arrived_mask = 0, gen = 0, alive_mask = 0, want_mask = 0;
  unsigned sync_gen = 0;       // completed __syncwarp()s of every live lane (memory ordering inside the warp)
  int op = -1;
};
thread_local std::vector<Warp> g_warps;

void yield_to_scheduler() { swapcontext(&g_fib[(size_t)g_cur].ctx, &g_main); }

void complete_collective(Warp& w) {
  const unsigned part = w.arrived_mask;
  switch (w.op) {
    case cuda_emu::OP_SYNCWARP: if (part == w.alive_mask) w.sync_gen++; break;   // shuffles and ballots order nothing
    case cuda_emu::OP_BALLOT: {
      unsigned b = 0;
      for (int l = 0; l < 32; ++l) if ((part >> l) & 1u) b |= (w.val[l] ? 1u : 0u) << l;
      for (int l = 0; l < 32; ++l) w.out[l] = b;
      break;
    }
    case cuda_emu::OP_SHFL_DOWN:
      for (int l = 0; l < 32; ++l) { const int s = l + w.arg[l]; w.out[l] = (s < 32 && ((part >> s) & 1u)) ? w.val[s] : w.val[l]; }
      break;
    case cuda_emu::OP_SHFL_UP:
      for (int l = 0; l < 32; ++l) { const int s = l - w.arg[l]; w.out[l] = (s >= 0 && ((part >> s) & 1u)) ? w.val[s] : w.val[l]; }
      break;
    case cuda_emu::OP_SHFL_XOR:
      for (int l = 0; l < 32; ++l) { const int s = l ^ w.arg[l]; w.out[l] = (s < 32 && ((part >> s) & 1u)) ? w.val[s] : w.val[l]; }
      break;
    case cuda_emu::OP_SHFL_IDX:
      for (int l = 0; l < 32; ++l) { const int s = w.arg[l] & 31; w.out[l] = ((part >> s) & 1u) ? w.val[s] : w.val[l]; }
      break;
    default: die("unknown collective");
  }
  w.arrived_mask = 0;
  w.op = -1;
  w.gen++;
  g_progress++;
}

// one warp instruction = the events of one warp with the same source line and occurrence number
void prof_reduce() {
  std::sort(g_prof_ev.begin(), g_prof_ev.end(), [](const ProfEv& a, const ProfEv& b) {
    const uint32_t wa = a.warp_lane >> 5, wb = b.warp_lane >> 5;
    if (wa != wb) return wa < wb;
    if (a.tuline != b.tuline) return a.tuline < b.tuline;
    if (a.write != b.write) return a.write < b.write;
    return a.occ < b.occ;
  });
  std::map<uint32_t, ProfAgg> local;
  std::vector<uint32_t> words;
  for (size_t i = 0; i < g_prof_ev.size();) {
    size_t j = i;
    words.clear();
    unsigned long long bytes = 0;
    while (j < g_prof_ev.size() && (g_prof_ev[j].warp_lane >> 5) == (g_prof_ev[i].warp_lane >> 5) && g_prof_ev[j].tuline == g_prof_ev[i].tuline &&
           g_prof_ev[j].write == g_prof_ev[i].write && g_prof_ev[j].occ == g_prof_ev[i].occ) {
      for (unsigned k = 0; k < g_prof_ev[j].nwords; ++k) words.push_back(g_prof_ev[j].word + k);
      bytes += 4ull * g_prof_ev[j].nwords;
      ++j;
    }
    std::sort(words.begin(), words.end());
    words.erase(std::unique(words.begin(), words.end()), words.end());
    unsigned per_bank[32] = {0}, wf = 0;
    for (uint32_t w : words) wf = std::max(wf, ++per_bank[w & 31u]);
    ProfAgg& a = local[(g_prof_ev[i].tuline << 1) | g_prof_ev[i].write];
    a.instr++; a.wavefronts += wf; a.ideal += (bytes + 127) / 128; a.lanes += (unsigned long long)(j - i);
    i = j;
  }
  g_prof_ev.clear();
  for (auto& m : g_prof_occ) m.clear();
  std::lock_guard<std::mutex> lk(g_prof_mu);
  for (auto& kv : local) { ProfAgg& g = g_prof[kv.first]; g.instr += kv.second.instr; g.wavefronts += kv.second.wavefronts; g.ideal += kv.second.ideal; g.lanes += kv.second.lanes; }
}

void prof_dump() {
  const char* path = prof_path();
  if (!path) return;
  FILE* f = fopen(path, "w");
  if (!f) return;
  std::lock_guard<std::mutex> lk(g_prof_mu);
  fprintf(f, "[");
  bool first = true;
  for (auto& kv : g_prof) {
    fprintf(f, "%s{\"tu\": %u, \"line\": %u, \"write\": %u, \"warp_instr\": %llu, \"wavefronts\": %llu, \"ideal\": %llu, \"lanes\": %llu}", first ? "" : ",\n ",
            (kv.first >> 1) >> 20, (kv.first >> 1) & 0xFFFFFu, kv.first & 1u, kv.second.instr, kv.second.wavefronts, kv.second.ideal, kv.second.lanes);
    first = false;
  }
  fprintf(f, "]\n");
  fclose(f);
}

void fiber_entry() {
  (*g_body)();
  Fiber& f = g_fib[(size_t)g_cur];
  if (!f.pending.empty()) die("thread exits with cp.async copies it never waited for");
  if (g_alive == 1 && !g_bulk.empty()) die("CTA exits with bulk copies nobody waited for");
  f.done = true;
  g_progress++;
  g_alive--;
  Warp& w = g_warps[(size_t)g_cur >> 5];
  w.alive_mask &= ~(1u << (g_cur & 31));
  // an exit may complete a rendezvous the others are waiting in
  if (g_bar_arrived > 0 && g_bar_arrived == g_alive) { g_bar_arrived = 0; g_bar_gen++; g_progress++; }
  if (w.arrived_mask && w.arrived_mask == (w.want_mask & w.alive_mask)) complete_collective(w);
  swapcontext(&f.ctx, &g_main);
  die("resumed a finished fiber");
}

void run_block() {
  const unsigned nt = g_nthreads;
  if (g_fib.size() < nt) g_fib.resize(nt);
  while (g_stack_pool.size() < nt) g_stack_pool.push_back((char*)malloc(STACK));
  g_warps.assign((nt + 31) / 32, Warp());
  for (unsigned i = 0; i < nt; ++i) {
    Fiber& f = g_fib[i];
    f.done = false; f.started = false; f.stack = g_stack_pool[i]; f.pending.clear();
    getcontext(&f.ctx);
    f.ctx.uc_stack.ss_sp = f.stack;
    f.ctx.uc_stack.ss_size = STACK;
    f.ctx.uc_link = &g_main;
    makecontext(&f.ctx, (void (*)())fiber_entry, 0);
    g_warps[i >> 5].alive_mask |= 1u << (i & 31);
  }
  g_alive = nt; g_bar_arrived = 0; g_bar_gen = 0;
  g_bulk.clear(); g_mbar.clear();
  if (race_on()) g_shadow.assign((g_dyn_bytes + 3) / 4, Shadow{Access{-1, 0, 0, 0, 0}, Access{-1, 0, 0, 0, 0}});
  else g_shadow.clear();
  // FTLM_EMU_ORDER: order in which runnable threads are resumed in every scheduling round - 0 ascending
  // (default), 1 descending, n >= 2 a fresh pseudo-random permutation per round (seed n).  A kernel whose
  // result depends on this order has a race (missing __syncthreads / __syncwarp); the tests run all three.
  static const int order_mode = getenv("FTLM_EMU_ORDER") ? atoi(getenv("FTLM_EMU_ORDER")) : 0;
  thread_local unsigned long long rng = 0x9E3779B97F4A7C15ull * (unsigned long long)(order_mode + 1);
  std::vector<unsigned> order(nt);
  for (unsigned i = 0; i < nt; ++i) order[i] = order_mode == 1 ? nt - 1 - i : i;
  for (;;) {
    const unsigned long long before = g_progress;
    bool any = false;
    if (order_mode >= 2)
      for (unsigned i = nt - 1; i > 0; --i) {
        rng ^= rng << 13; rng ^= rng >> 7; rng ^= rng << 17;
        std::swap(order[i], order[(unsigned)(rng % (i + 1))]);
      }
    for (unsigned oi = 0; oi < nt; ++oi) {
      const unsigned i = order[oi];
      Fiber& f = g_fib[i];
      if (f.done) continue;
      any = true;
      g_cur = (int)i;
      threadIdx.x = i; threadIdx.y = 0; threadIdx.z = 0;
      if (!f.started) { f.started = true; g_progress++; }
      swapcontext(&g_main, &f.ctx);
    }
    if (!any) break;
    if (g_progress == before) die("deadlock: no thread of the CTA can make progress (mismatched barrier / collective)");
  }
  g_cur = -1;
  if (prof_path()) prof_reduce();
}

cudaError_t g_last = cudaSuccess;

}  // namespace

namespace cuda_emu {

unsigned char* dyn_smem() { return g_dyn; }

void cp_async_issue(void* smem_dst, const void* gsrc, size_t bytes) {
  if (g_cur < 0) die("cp.async outside a kernel");
  if (bytes != 4 && bytes != 8 && bytes != 16) die("cp.async copies 4, 8 or 16 bytes");
  if (((uintptr_t)smem_dst % bytes) || ((uintptr_t)gsrc % bytes)) die("cp.async: misaligned source or destination");
  PendingCopy c;
  c.dst = smem_dst; c.bytes = bytes;
  memcpy(c.data, gsrc, bytes);              // faults here if the source is out of range (guard page)
  memset(smem_dst, 0xFF, bytes);            // not visible yet: NaN until the issuing thread waits
  g_fib[(size_t)g_cur].pending.push_back(c);
}

void cp_async_wait_all() {
  if (g_cur < 0) die("cp.async.wait_all outside a kernel");
  Fiber& f = g_fib[(size_t)g_cur];
  for (const PendingCopy& c : f.pending) { smem_access(c.dst, c.bytes, true, 0, 0); memcpy(c.dst, c.data, c.bytes); }
  f.pending.clear();
}

// ---- bulk copies + mbarriers (per CTA = per host thread) ------------------------------------------------------------
void mbar_init(void* mbar, int count) {
  if (g_cur < 0) die("mbarrier.init outside a kernel");
  MBar b; b.count = count; b.pending = count;
  g_mbar[mbar] = b;
}

void mbar_arrive_expect_tx(void* mbar, unsigned bytes) {
  auto it = g_mbar.find(mbar);
  if (it == g_mbar.end()) die("mbarrier.arrive on an uninitialised barrier");
  it->second.tx += (long)bytes;
  if (--it->second.pending < 0) die("mbarrier: more arrivals than its count");
  g_progress++;
}

void bulk_issue(void* smem_dst, const void* gsrc, unsigned bytes, void* mbar, int tu, int line) {
  if (g_cur < 0) die("cp.async.bulk outside a kernel");
  if (bytes == 0 || (bytes & 15u) || ((uintptr_t)smem_dst & 15u) || ((uintptr_t)gsrc & 15u)) die("cp.async.bulk: size, source and destination must be multiples of 16 bytes");
  if ((unsigned char*)smem_dst < g_dyn || (unsigned char*)smem_dst + bytes > g_dyn + g_dyn_bytes) die("cp.async.bulk: destination outside the dynamic shared memory");
  if (g_mbar.find(mbar) == g_mbar.end()) die("cp.async.bulk on an uninitialised barrier");
  PendingBulk c;
  c.dst = smem_dst; c.mbar = mbar;
  c.data.assign((const unsigned char*)gsrc, (const unsigned char*)gsrc + bytes);    // faults here if the source is out of range
  smem_access(smem_dst, bytes, true, tu, line);                                      // overwriting what others may still read?
  memset(smem_dst, 0xFF, bytes);
  g_bulk.push_back(std::move(c));
}

void mbar_wait(void* mbar, unsigned parity) {
  if (g_cur < 0) die("mbarrier.try_wait outside a kernel");
  for (;;) {
    auto it = g_mbar.find(mbar);
    if (it == g_mbar.end()) die("mbarrier.try_wait on an uninitialised barrier");
    MBar& b = it->second;
    if ((b.completed & 1u) != (parity & 1u)) return;           // the phase of this parity has completed
    if (b.pending == 0) {                                      // all arrivals made: the outstanding copies complete now
      for (size_t k = 0; k < g_bulk.size();) {
        if (g_bulk[k].mbar != mbar) { ++k; continue; }
        PendingBulk& c = g_bulk[k];
        memcpy(c.dst, c.data.data(), c.data.size());
        b.tx -= (long)c.data.size();
        const size_t w0 = (size_t)((unsigned char*)c.dst - g_dyn) / 4, w1 = w0 + c.data.size() / 4;
        for (size_t w = w0; w < w1 && w < g_shadow.size(); ++w) { g_shadow[w].w.tid = -1; g_shadow[w].r.tid = -1; }   // written by the async proxy
        g_bulk.erase(g_bulk.begin() + (long)k);
      }
      if (b.tx != 0) die("mbarrier: expected and completed transaction bytes differ");
      b.completed++; b.pending = b.count;
      g_progress++;
      continue;
    }
    yield_to_scheduler();
    threadIdx.x = (unsigned)g_cur;
  }
}

void smem_skip(int tu, int line) {
  if (g_cur < 0 || !prof_path()) return;
  if (g_prof_occ.size() < g_nthreads) g_prof_occ.resize(g_nthreads);
  g_prof_occ[(size_t)g_cur][((uint32_t)tu << 20) | (uint32_t)line]++;
}

bool smem_access(const void* p, size_t bytes, bool write, int tu, int line) {
  if (g_cur < 0 || g_shadow.empty()) return true;
  const unsigned char* a = (const unsigned char*)p;
  if (a < g_dyn || a >= g_dyn + g_dyn_bytes) return true;            // static __shared__ variables, global memory
  if (prof_path() && (tu || line)) {
    const uint32_t key = ((uint32_t)tu << 20) | (uint32_t)line;
    if (g_prof_occ.size() < g_nthreads) g_prof_occ.resize(g_nthreads);
    const uint32_t occ = g_prof_occ[(size_t)g_cur][key]++;
    g_prof_ev.push_back(ProfEv{(uint32_t)g_cur, key, occ, (uint32_t)((a - g_dyn) / 4), (uint8_t)((bytes + 3) / 4), (uint8_t)write});
  }
  const int t = g_cur;
  const unsigned bar = g_bar_gen, wgen = g_warps[(size_t)t >> 5].sync_gen;
  auto ordered = [&](const Access& x) {
    if (x.tid < 0 || x.tid == t) return true;
    if (x.bar != bar) return true;                                    // a __syncthreads completed in between
    return (x.tid >> 5) == (t >> 5) && x.wgen != wgen;                // same warp and a __syncwarp in between
  };
  const size_t w0 = (size_t)(a - g_dyn) / 4, w1 = ((size_t)(a - g_dyn) + bytes - 1) / 4;
  for (size_t k = w0; k <= w1 && k < g_shadow.size(); ++k) {
    Shadow& sh = g_shadow[k];
    const Access* bad = nullptr;
    const char* kind = "";
    if (!ordered(sh.w)) { bad = &sh.w; kind = write ? "write after write" : "read after write"; }
    else if (write && !ordered(sh.r)) { bad = &sh.r; kind = "write after read"; }
    if (bad) {
      fprintf(stderr, "cuda_emu: shared-memory race (%s) on dynamic smem byte %zu: thread %d (tu %d line %d) and thread %d (tu %d line %d) "
              "with no __syncthreads%s between them (block %u)\n", kind, k * 4, bad->tid, bad->tu, bad->line, t, tu, line,
              (bad->tid >> 5) == (t >> 5) ? " / __syncwarp" : "", blockIdx.x);
      fflush(stderr);
      abort();
    }
    if (write) { sh.w = Access{t, bar, wgen, tu, line}; sh.r.tid = -1; }
    else sh.r = Access{t, bar, wgen, tu, line};
  }
  return true;
}

void sync_threads() {
  if (g_cur < 0) die("__syncthreads outside a kernel");
  const unsigned my = g_bar_gen;
  g_bar_arrived++;
  if (g_bar_arrived == g_alive) { g_bar_arrived = 0; g_bar_gen++; g_progress++; return; }
  while (g_bar_gen == my) yield_to_scheduler();
  threadIdx.x = (unsigned)g_cur;
}

uint64_t collective(int op, unsigned mask, uint64_t v, int arg) {
  if (g_cur < 0) die("warp collective outside a kernel");
  Warp& w = g_warps[(size_t)g_cur >> 5];
  const int lane = g_cur & 31;
  if (!((mask >> lane) & 1u)) die("warp collective: calling lane not in its own mask");
  if (w.arrived_mask == 0) { w.op = op; w.want_mask = mask; }
  else if (w.op != op || w.want_mask != mask) die("warp collective mismatch: lanes of one warp are in different collectives");
  w.val[lane] = v; w.arg[lane] = arg;
  w.arrived_mask |= 1u << lane;
  const unsigned my = w.gen;
  if (w.arrived_mask == (w.want_mask & w.alive_mask)) complete_collective(w);
  else while (w.gen == my) yield_to_scheduler();
  threadIdx.x = (unsigned)g_cur;
  return w.out[lane];
}

void launch(unsigned grid, unsigned block, size_t dyn_bytes, const std::function<void()>& body) {
  if (g_cur >= 0) die("nested launch");
  static const bool prof_registered = (prof_path() ? atexit(prof_dump) : 0, true);
  (void)prof_registered;
  if (grid == 0 || block == 0 || block > 1024) { g_last = cudaErrorInvalidValue; return; }
  if (dyn_bytes > 227 * 1024) { g_last = cudaErrorInvalidValue; return; }
  // CTAs are taken from a shared counter by a few host threads and run concurrently (one CTA in flight per host
  // thread, its CUDA threads as fibers on that thread)
  static const unsigned max_workers = getenv("FTLM_EMU_CTAS") ? (unsigned)std::max(1, atoi(getenv("FTLM_EMU_CTAS"))) : 4u;
  std::atomic<unsigned> next{0};
  auto worker = [&]() {
    {
      std::lock_guard<std::mutex> lk(g_stack_mu);
      if (g_stack_pool.empty() && !g_free_stack_sets.empty()) { g_stack_pool.swap(g_free_stack_sets.back()); g_free_stack_sets.pop_back(); }
    }
    g_body = &body;
    g_nthreads = block;
    gridDim = dim3(grid); blockDim = dim3(block);
    for (;;) {
      const unsigned b = next.fetch_add(1);
      if (b >= grid) break;
      blockIdx.x = b; blockIdx.y = 0; blockIdx.z = 0;
      g_dyn = dyn_bytes ? (unsigned char*)guarded_alloc(dyn_bytes) : nullptr;
      g_dyn_bytes = dyn_bytes;
      run_block();
      if (g_dyn) guarded_free(g_dyn);
      g_dyn = nullptr; g_dyn_bytes = 0;
    }
    g_body = nullptr;
    g_fib.clear(); g_warps.clear(); g_shadow.clear();
    std::lock_guard<std::mutex> lk(g_stack_mu);
    g_free_stack_sets.emplace_back();
    g_free_stack_sets.back().swap(g_stack_pool);
  };
  const unsigned nw = std::min(grid, max_workers);
  if (nw <= 1) { worker(); return; }
  std::vector<std::thread> pool;
  for (unsigned k = 0; k < nw; ++k) pool.emplace_back(worker);
  for (std::thread& th : pool) th.join();
}

}  // namespace cuda_emu

// ---- runtime API ---------------------------------------------------------------------------------
struct cuda_emu_event { double t_ms; };

cudaError_t cudaGetDeviceCount(int* n) { *n = getenv("FTLM_EMU_NO_DEVICE") ? 0 : 1; return *n ? cudaSuccess : cudaErrorNoDevice; }
cudaError_t cudaSetDevice(int) { return cudaSuccess; }
cudaError_t cudaGetDeviceProperties(cudaDeviceProp* p, int) {
  memset(p, 0, sizeof(*p));
  snprintf(p->name, sizeof(p->name), "cuda_emu (host SIMT emulation)");
  const char* s = getenv("FTLM_EMU_SMS");
  p->multiProcessorCount = s ? atoi(s) : 3;
  p->sharedMemPerBlockOptin = 227 * 1024;
  p->major = 10; p->minor = 0;
  p->l2CacheSize = 126u << 20;
  return cudaSuccess;
}
cudaError_t cudaMalloc(void** p, size_t bytes) {
  *p = guarded_alloc(bytes ? bytes : 16);
  if (!*p) { g_last = cudaErrorMemoryAllocation; return cudaErrorMemoryAllocation; }
  return cudaSuccess;
}
cudaError_t cudaFree(void* p) { if (p) guarded_free(p); return cudaSuccess; }
cudaError_t cudaMemcpy(void* d, const void* s, size_t n, cudaMemcpyKind) { if (n) memmove(d, s, n); return cudaSuccess; }
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind k, cudaStream_t) { return cudaMemcpy(d, s, n, k); }
cudaError_t cudaMemset(void* p, int v, size_t n) { if (n) memset(p, v, n); return cudaSuccess; }
cudaError_t cudaMemsetAsync(void* p, int v, size_t n, cudaStream_t) { return cudaMemset(p, v, n); }
cudaError_t cudaGetLastError() { cudaError_t e = g_last; g_last = cudaSuccess; return e; }
cudaError_t cudaPeekAtLastError() { return g_last; }
const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : e == cudaErrorMemoryAllocation ? "out of memory" : "cuda_emu error"; }
cudaError_t cudaDeviceSynchronize() { return cudaSuccess; }
cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
static double now_ms() { timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts); return ts.tv_sec * 1e3 + ts.tv_nsec * 1e-6; }
cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = new cuda_emu_event{0.0}; return cudaSuccess; }
cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t) { e->t_ms = now_ms(); return cudaSuccess; }
cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) { *ms = (float)(b->t_ms - a->t_ms); return cudaSuccess; }
