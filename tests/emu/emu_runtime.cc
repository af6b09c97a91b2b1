// emu_runtime.cc -- TEST INFRASTRUCTURE ONLY (see emu_core.h): fiber scheduler, models of the asynchronous hardware
// units, and a stand-in for the CUDA runtime API that EXECUTES kernel launches on the host.
//
// Linked with the g++-compiled product sources into tests/emu/_build/libgmco_emu.so.  Nothing here computes a step of
// the method: it moves bytes (TMA), multiplies the operand tiles a kernel's descriptors point at (tcgen05.mma) and keeps
// the synchronisation objects' state.  What a kernel asks of it is checked: shared-memory window, TMEM allocation,
// device allocations, descriptor fields, alignment rules, barrier over-arrival, work left in flight at exit.
#include "emu_core.h"

#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <time.h>

#include <deque>
#include <array>
#include <map>
#include <memory>
#include <string>
#include <unordered_map>
#include <vector>

#if defined(__SANITIZE_ADDRESS__)
#include <sanitizer/asan_interface.h>
#include <sanitizer/common_interface_defs.h>
#define EMU_ASAN 1
#else
#define EMU_ASAN 0
#endif

namespace emu {

// ------------------------------------------------------------------------------------------------------------------
// configuration and records (read and written through the emu_* C functions at the end of this file)
struct Config {
  uint64_t seed = 1;
  int max_delay = 400;          // asynchronous operations complete 1 .. max_delay scheduler ticks after issue
  int mma_delay = -1;           // >= 0: the tensor pipe's own bound (a slow pipe exposes ring slots refilled too early,
                                // a fast one with slow copies exposes operands read before they landed)
  int dyn_misalign = 16;        // window offset of dynamic shared memory = 1024 + this (the kernels align by hand)
  int sm_count = 148;
  long drop_tma = -1;           // fault injection: the n-th TMA load (0-based, per process) never completes
  long drop_commit = -1;        // fault injection: the n-th tcgen05.commit never arrives
  int shuffle = 1;              // randomise the order in which the fibers of a CTA are resumed
  unsigned starve_mask = 0;     // warps (bit = warp index) that only get a turn every starve_period-th round: a slow
  int starve_period = 1;        // producer, issuer or epilogue must change nothing but the time it takes
  int verbose = 0;
};
static Config g_cfg;
static int g_violations;
static char g_violation_msg[1024];
static long g_tma_count, g_commit_count, g_mma_count, g_hangs;
// per kernel: bytes landed in shared memory by TMA / bulk copies, bytes of shared memory read by MMA operands, tensor-pipe
// cycles x SMs (a kind::tf32 MMA of N columns keeps each SM it runs on busy for N / 2 cycles: profiles/r1_mma_rate.md)
static std::map<std::string, std::array<long, 3>> g_traffic;
struct LaunchRec { std::string name; dim3 grid, block; size_t smem; int captured; };
static std::vector<LaunchRec> g_launches;
static std::map<std::string, long> g_kernel_runs;
static std::map<std::string, double> g_kernel_secs;      // host seconds spent emulating each kernel          // executions (outside capture + graph replays) by kernel name
static cudaError_t g_last_error = cudaSuccess, g_sticky = cudaSuccess;

void violation(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  if (!g_violations) {
    vsnprintf(g_violation_msg, sizeof g_violation_msg, fmt, ap);
    if (g_cfg.verbose) fprintf(stderr, "[emu] violation: %s\n", g_violation_msg);
  }
  va_end(ap);
  g_violations++;
}

// ------------------------------------------------------------------------------------------------------------------
// device memory: host allocations with a table for range checks
struct Alloc { char* p; size_t n; };
static std::vector<Alloc> g_allocs;
static const Alloc* find_alloc(const void* p) {
  for (const Alloc& a : g_allocs)
    if (a.p && (const char*)p >= a.p && (const char*)p < a.p + a.n) return &a;
  return nullptr;
}
static bool in_device(const void* p, size_t n) {
  const Alloc* a = find_alloc(p);
  return a && (const char*)p + n <= a->p + a->n;
}

// ------------------------------------------------------------------------------------------------------------------
// fibers
extern "C" void emu_switch(void** save_sp, void* load_sp);
asm(R"(
.text
.globl emu_switch
.type emu_switch,@function
emu_switch:
  pushq %rbp
  pushq %rbx
  pushq %r12
  pushq %r13
  pushq %r14
  pushq %r15
  movq %rsp, (%rdi)
  movq %rsi, %rsp
  popq %r15
  popq %r14
  popq %r13
  popq %r12
  popq %rbx
  popq %rbp
  ret
.size emu_switch,.-emu_switch
)");

constexpr size_t kStackBytes = 192 * 1024;
struct Gang;
struct Fiber {
  void* sp = nullptr;
  char* stack = nullptr;
  bool done = false;
  ThreadCtx ctx{};
  int bulk_pending = 0;         // bulk stores of this thread whose shared-memory source has not been read yet
  const char* where = "running"; // what the thread last blocked on (reported when a CTA hangs)
  uint32_t where_arg = 0;
  Gang* gang = nullptr;
};
thread_local ThreadCtx* g_cur = nullptr;
static Fiber* g_fiber = nullptr;
static void* g_sched_sp = nullptr;
static std::vector<char*> g_stack_pool;

static char* get_stack() {
  if (!g_stack_pool.empty()) { char* s = g_stack_pool.back(); g_stack_pool.pop_back(); return s; }
  void* p = nullptr;
  if (posix_memalign(&p, 64, kStackBytes)) abort();
  return (char*)p;
}

struct Warp {
  unsigned live = 0, arrived = 0, mask = 0xffffffffu;
  uint32_t gen = 0;
  uint64_t xbuf[2][32];
  unsigned ballot[2] = {0, 0};
};
struct Mbar { uint32_t expected = 0, pending = 0; int64_t tx = 0; uint32_t phase = 0; };

constexpr int kTmemLanes = 128, kTmemCols = 512;
constexpr uint32_t kDynWindowBase = 1024;
constexpr size_t kWindowBytes = 1u << 18;

struct Cta {
  int rank = 0;
  uint3 bid{};
  uint8_t* region = nullptr;      // 256 KB, 256 KB-aligned: host address bits [0, 18) = window offset, as on the hardware
  uint8_t* dyn = nullptr;
  size_t dyn_bytes = 0;
  uint32_t dyn_base = kDynWindowBase;
  std::unordered_map<uint32_t, Mbar> mbars;               // by window offset
  std::vector<const void*> statics;                         // 8-byte granules of static shared memory that were given a window address
  std::vector<uint32_t> tmem;                               // [128][512]
  bool tmem_allocated = false;
  uint32_t tmem_cols = 0;
  int nthreads = 0, live = 0;
  int bar_arrived = 0;
  uint32_t bar_gen = 0;
  std::vector<Warp> warps;
  Gang* gang = nullptr;
};

// What an operation in flight will touch, for the hazard checks made when OTHER operations are issued: a correct kernel
// orders them through its barriers, so an overlap found at issue time is a protocol error whatever the timing.
struct Range { const Cta* cta; uint32_t lo, hi; };             // shared-memory window addresses [lo, hi) of one CTA
struct Cols { const Cta* cta; uint32_t lo, hi; };              // TMEM columns [lo, hi) of one CTA (all 128 lanes)
struct Touch { std::vector<Range> smem_w, smem_r; std::vector<Cols> tmem_w, tmem_r; };
struct Op { uint64_t due; std::function<void()> fn; Touch touch; };

struct Gang {
  std::vector<std::unique_ptr<Cta>> ctas;
  std::vector<std::unique_ptr<Fiber>> fibers;
  const std::function<void()>* body = nullptr;
  int live = 0;
  int cl_arrived = 0;
  uint32_t cl_gen = 0;
  uint64_t tick = 0, progress = 0;
  uint64_t vtime_jump = 0;
  std::deque<Op> ops;                 // unordered units (TMA, bulk copies)
  std::deque<Op> pipe;                // the tensor pipe of the gang: in order
  uint64_t pipe_last_due = 0;
  uint64_t rng = 88172645463325252ull;
  const char* kernel = "";
  bool hung = false;
};
static Gang* g_gang = nullptr;

static uint64_t rnd(Gang* g) { uint64_t x = g->rng; x ^= x << 13; x ^= x >> 7; x ^= x << 17; g->rng = x; return x; }
static uint64_t delay(Gang* g) { return 1 + (g_cfg.max_delay > 1 ? rnd(g) % (uint64_t)g_cfg.max_delay : 0); }

void note_progress() { if (g_gang) g_gang->progress++; }

static void switch_to_scheduler() {
  Fiber* f = g_fiber;
#if EMU_ASAN
  void* fake = nullptr;
  __sanitizer_start_switch_fiber(f->done ? nullptr : &fake, nullptr, 0);
#endif
  emu_switch(&f->sp, g_sched_sp);
#if EMU_ASAN
  __sanitizer_finish_switch_fiber(fake, nullptr, nullptr);
#endif
}
void yield() { switch_to_scheduler(); }

static void warp_try_release(Warp& w) {
  const unsigned need = w.mask & w.live;
  if (w.arrived && (w.arrived & need) == need) {
    w.arrived = 0; w.gen++;
    w.ballot[w.gen & 1] = 0;
    note_progress();
  }
}
static void cta_try_release(Cta* c) {
  if (c->bar_arrived > 0 && c->bar_arrived >= c->live) { c->bar_arrived = 0; c->bar_gen++; note_progress(); }
}
static void cluster_try_release(Gang* g) {
  if (g->cl_arrived > 0 && g->cl_arrived >= g->live) { g->cl_arrived = 0; g->cl_gen++; note_progress(); }
}

static void fiber_main() {
#if EMU_ASAN
  __sanitizer_finish_switch_fiber(nullptr, nullptr, nullptr);
#endif
  Fiber* f = g_fiber;
  (*f->gang->body)();
  // thread exit: it no longer takes part in any barrier
  f = g_fiber;
  f->done = true;
  Cta* c = f->ctx.cta;
  Gang* g = f->gang;
  if (f->bulk_pending) violation("%s: a thread left the kernel with %d bulk stores still reading shared memory", g->kernel, f->bulk_pending);
  c->live--; g->live--;
  Warp& w = c->warps[f->ctx.warp];
  w.live &= ~(1u << f->ctx.lane);
  warp_try_release(w);
  cta_try_release(c);
  cluster_try_release(g);
  note_progress();
  switch_to_scheduler();
  abort();   // never resumed
}

static void make_fiber(Fiber* f) {
  f->stack = get_stack();
  uintptr_t top = ((uintptr_t)f->stack + kStackBytes) & ~(uintptr_t)15;
  // after the six pops and the ret of emu_switch the stack pointer must be 8 mod 16, as at any function entry
  uint64_t* sp = (uint64_t*)top;
  *--sp = 0;                                // would-be return address of fiber_main (never used)
  *--sp = (uint64_t)(uintptr_t)&fiber_main;
  for (int i = 0; i < 6; ++i) *--sp = 0;
  f->sp = sp;
}

static void resume(Fiber* f) {
  g_fiber = f; g_cur = &f->ctx;
#if EMU_ASAN
  void* fake = nullptr;
  __sanitizer_start_switch_fiber(&fake, f->stack, kStackBytes);
#endif
  emu_switch(&g_sched_sp, f->sp);
#if EMU_ASAN
  __sanitizer_finish_switch_fiber(fake, nullptr, nullptr);
#endif
  g_fiber = nullptr; g_cur = nullptr;
}

static void run_due(Gang* g) {
  // unordered units: anything that is due; tensor pipe: in order
  for (size_t i = 0; i < g->ops.size();) {
    if (g->ops[i].due <= g->tick) {
      auto fn = std::move(g->ops[i].fn);
      g->ops.erase(g->ops.begin() + (long)i);
      fn(); g->progress++;
    } else ++i;
  }
  while (!g->pipe.empty() && g->pipe.front().due <= g->tick) {
    auto fn = std::move(g->pipe.front().fn);
    g->pipe.pop_front();
    fn(); g->progress++;
  }
}
static void post(Gang* g, std::function<void()> fn, Touch touch = Touch()) { g->ops.push_back(Op{g->tick + delay(g), std::move(fn), std::move(touch)}); }
static void post_pipe(Gang* g, std::function<void()> fn, Touch touch = Touch()) {
  const int md = g_cfg.mma_delay >= 0 ? g_cfg.mma_delay : g_cfg.max_delay;
  uint64_t due = g->tick + 1 + (md > 1 ? rnd(g) % (uint64_t)md : 0);
  if (due < g->pipe_last_due) due = g->pipe_last_due;
  g->pipe_last_due = due;
  g->pipe.push_back(Op{due, std::move(fn), std::move(touch)});
}

static bool overlaps(const std::vector<Range>& a, const Cta* c, uint32_t lo, uint32_t hi) {
  for (const Range& r : a) if (r.cta == c && r.lo < hi && lo < r.hi) return true;
  return false;
}
static bool overlaps(const std::vector<Cols>& a, const Cta* c, uint32_t lo, uint32_t hi) {
  for (const Cols& r : a) if (r.cta == c && r.lo < hi && lo < r.hi) return true;
  return false;
}
// an asynchronous WRITE of shared memory [lo, hi) is being issued: nothing in flight may still read or write it
static void check_smem_write_issue(Gang* g, const Cta* c, uint32_t lo, uint32_t hi, const char* what) {
  for (const Op& o : g->pipe)
    if (overlaps(o.touch.smem_r, c, lo, hi)) { violation("%s: %s into shared memory [0x%x, 0x%x) while MMAs that read it are still in flight (slot refilled before its consumer's commit)", g->kernel, what, lo, hi); return; }
  for (const Op& o : g->ops)
    if (overlaps(o.touch.smem_w, c, lo, hi)) { violation("%s: %s into shared memory [0x%x, 0x%x) while another copy into it is still in flight", g->kernel, what, lo, hi); return; }
}
// an MMA that READS shared memory [lo, hi) is being issued: every copy into it must have landed
static void check_smem_read_issue(Gang* g, const Cta* c, uint32_t lo, uint32_t hi, const char* what) {
  for (const Op& o : g->ops)
    if (overlaps(o.touch.smem_w, c, lo, hi)) { violation("%s: %s reads shared memory [0x%x, 0x%x) while a copy into it is still in flight (issued before the full barrier)", g->kernel, what, lo, hi); return; }
}
// a thread reads / writes TMEM columns: no MMA in flight may write (read: or read) them
static void check_tmem_thread_access(Gang* g, const Cta* c, uint32_t lo, uint32_t hi, bool write, const char* what) {
  for (const Op& o : g->pipe) {
    if (overlaps(o.touch.tmem_w, c, lo, hi)) { violation("%s: %s of TMEM columns [%u, %u) while MMAs that write them are in flight (accumulator touched before its commit arrived)", g->kernel, what, lo, hi); return; }
    if (write && overlaps(o.touch.tmem_r, c, lo, hi)) { violation("%s: %s of TMEM columns [%u, %u) while MMAs that read them as an operand are in flight", g->kernel, what, lo, hi); return; }
  }
}
#if EMU_ASAN
// while a copy into shared memory is in flight the kernel's own loads and stores must stay away from its destination
static void asan_guard(Cta* c, uint32_t addr, size_t bytes, bool on) {
  const uint32_t off = addr & 0xffffffu;
  if (off < c->dyn_base || (size_t)off + bytes > (size_t)c->dyn_base + c->dyn_bytes) return;
  if (on) __asan_poison_memory_region(c->dyn + (off - c->dyn_base), bytes);
  else __asan_unpoison_memory_region(c->dyn + (off - c->dyn_base), bytes);
}
#else
static void asan_guard(Cta*, uint32_t, size_t, bool) {}
#endif

unsigned long long virtual_ns() { return g_gang ? 1000000ull + g_gang->tick * 20ull + g_gang->vtime_jump : 0ull; }
void sleep_ns(unsigned ns) {
  if (!g_gang) return;
  const uint64_t until = g_gang->tick + ns / 20 + 1;
  while (g_gang->tick < until) yield();
}

static void run_gang(Gang* g) {
  g_gang = g;
  std::vector<Fiber*> order;
  for (auto& f : g->fibers) order.push_back(f.get());
  long stagnant = 0;
  uint64_t round = 0;
  while (g->live > 0) {
    const uint64_t p0 = g->progress;
    if (g_cfg.shuffle && order.size() > 1) {
      // rotate the starting point and swap a few entries: cheap, seeded, enough to vary the interleaving
      const size_t r = rnd(g) % order.size();
      std::rotate(order.begin(), order.begin() + (long)r, order.end());
      for (int i = 0; i < 4; ++i) std::swap(order[rnd(g) % order.size()], order[rnd(g) % order.size()]);
    }
    const bool full_round = g_cfg.starve_period <= 1 || (++round % (uint64_t)g_cfg.starve_period) == 0;
    for (Fiber* f : order) {
      if (f->done) continue;
      if (!full_round && ((g_cfg.starve_mask >> (f->ctx.warp & 31)) & 1u)) continue;
      resume(f);
      g->tick++;
      run_due(g);
    }
    if (g->progress != p0) { stagnant = 0; continue; }
    if (!full_round) continue;                      // only a round in which every thread had its turn can show a standstill
    if (!g->ops.empty() || !g->pipe.empty()) {      // everybody waits for a hardware unit: let its time come
      uint64_t next = ~0ull;
      for (const Op& o : g->ops) next = std::min(next, o.due);
      if (!g->pipe.empty()) next = std::min(next, g->pipe.front().due);
      if (next > g->tick) g->tick = next;
      run_due(g);
      stagnant = 0;
      continue;
    }
    // nothing moves and nothing is in flight: on the hardware this is a hang.  Let (virtual) time pass so that bounded
    // waits run into their limit; waits without a bound never will, and the launch is then abandoned.
    if (++stagnant >= 3) g->vtime_jump += 250000000ull;
    if (stagnant > 120000) {
      g->hung = true; g_hangs++;
      if (g_cfg.verbose) {
        std::map<std::string, int> stuck;
        for (auto& f : g->fibers)
          if (!f->done) { char b[160]; snprintf(b, sizeof b, "cta %d warp %d: %s 0x%x", f->ctx.cta->rank, f->ctx.warp, f->where, f->where_arg); stuck[b]++; }
        for (auto& kv : stuck) fprintf(stderr, "[emu] stuck: %3d threads  %s\n", kv.second, kv.first.c_str());
      }
      violation("%s: CTA (%u,%u) hangs: no thread can make progress and nothing is in flight", g->kernel,
                g->ctas[0]->bid.x, g->ctas[0]->bid.y);
      break;
    }
  }
  if (!g->hung) {
    if (!g->ops.empty() || !g->pipe.empty())
      violation("%s: CTA (%u,%u) ended with %zu asynchronous operations still in flight", g->kernel, g->ctas[0]->bid.x,
                g->ctas[0]->bid.y, g->ops.size() + g->pipe.size());
    for (auto& c : g->ctas)
      if (c->tmem_allocated) violation("%s: CTA (%u,%u) ended without tcgen05.dealloc", g->kernel, c->bid.x, c->bid.y);
  }
  for (auto& f : g->fibers) { g_stack_pool.push_back(f->stack); f->stack = nullptr; }
  g_gang = nullptr;
}

// ------------------------------------------------------------------------------------------------------------------
// barriers of the SIMT model
void cta_barrier() {
  Cta* c = cur()->cta;
  const uint32_t gen = c->bar_gen;
  c->bar_arrived++;
  cta_try_release(c);
  g_fiber->where = "__syncthreads"; g_fiber->where_arg = 0;
  while (c->bar_gen == gen) yield();
}
void cluster_barrier() {
  Gang* g = g_gang;
  const uint32_t gen = g->cl_gen;
  g->cl_arrived++;
  cluster_try_release(g);
  g_fiber->where = "cluster barrier"; g_fiber->where_arg = 0;
  while (g->cl_gen == gen) yield();
}
void warp_barrier(unsigned mask) {
  ThreadCtx* t = cur();
  Warp& w = t->cta->warps[t->warp];
  if (!(mask & (1u << t->lane))) { violation("%s: warp-synchronous operation whose mask omits the calling lane", g_gang->kernel); return; }
  const uint32_t gen = w.gen;
  w.mask = mask;
  w.arrived |= 1u << t->lane;
  warp_try_release(w);
  g_fiber->where = "warp-synchronous operation (arrived mask in arg)"; g_fiber->where_arg = w.arrived;
  while (w.gen == gen) yield();
}
void warp_exchange(unsigned mask, const void* in, void* out, int bytes, int src_lane) {
  ThreadCtx* t = cur();
  Warp& w = t->cta->warps[t->warp];
  const int par = (int)(w.gen & 1);
  // (checked on entry: once the barrier below has released, faster lanes may already have left the kernel)
  const bool src_ok = (w.live & mask & (1u << src_lane)) != 0;
  memcpy(&w.xbuf[par][t->lane], in, (size_t)bytes);
  warp_barrier(mask);
  if (!src_ok) {
    // reading a lane that does not take part: undefined on the hardware
    violation("%s: shuffle reads lane %d, which is not a live lane of the mask", g_gang->kernel, src_lane);
    memcpy(out, in, (size_t)bytes);
    return;
  }
  memcpy(out, &w.xbuf[par][src_lane], (size_t)bytes);
}
unsigned warp_ballot(unsigned mask, int pred) {
  ThreadCtx* t = cur();
  Warp& w = t->cta->warps[t->warp];
  const int par = (int)(w.gen & 1);
  if (pred) w.ballot[par] |= 1u << t->lane;
  warp_barrier(mask);
  return w.ballot[par] & mask;
}
bool elect_one_sync() {
  ThreadCtx* t = cur();
  Warp& w = t->cta->warps[t->warp];
  const int leader = __builtin_ctz(w.live);    // on entry: after the barrier faster lanes may already have left the kernel
  warp_barrier(0xffffffffu);
  return t->lane == leader;
}

// ------------------------------------------------------------------------------------------------------------------
// shared-memory window.  A shared::cta address is an offset into the CTA's window; bits 24.. hold (rank + 1) for an
// address that mapa produced (shared::cluster), 0 for "this CTA".
void* dyn_smem_ptr() { return cur()->cta->dyn; }
uint32_t dynamic_smem_bytes() { return (uint32_t)cur()->cta->dyn_bytes; }

uint32_t smem_window_addr(const void* p) {
  Cta* c = cur()->cta;
  const uint8_t* q = (const uint8_t*)p;
  if (q >= c->dyn && q < c->dyn + c->dyn_bytes) return c->dyn_base + (uint32_t)(q - c->dyn);
  // static shared memory (only 8-byte objects such as mbarriers are ever addressed this way)
  const void* granule = (const void*)((uintptr_t)p & ~(uintptr_t)7);
  for (size_t i = 0; i < c->statics.size(); ++i)
    if (c->statics[i] == granule) return 16 + 8 * (uint32_t)i + (uint32_t)((uintptr_t)p & 7);
  if (16 + 8 * c->statics.size() + 8 > kDynWindowBase) { violation("%s: too many static shared objects addressed", g_gang->kernel); return 0; }
  c->statics.push_back(granule);
  return 16 + 8 * (uint32_t)(c->statics.size() - 1) + (uint32_t)((uintptr_t)p & 7);
}
uint32_t cluster_rank() { return (uint32_t)cur()->cta->rank; }
uint32_t map_to_rank(uint32_t addr, uint32_t rank) { return (addr & 0xffffffu) | ((rank + 1) << 24); }

static Cta* owner_of(uint32_t addr, Cta* self) {
  const uint32_t r = addr >> 24;
  if (r == 0) return self;
  Gang* g = self->gang;
  if (r - 1 >= g->ctas.size()) { violation("%s: shared::cluster address 0x%x names CTA rank %u of a cluster of %zu", g->kernel, addr, r - 1, g->ctas.size()); return nullptr; }
  return g->ctas[r - 1].get();
}
// host pointer of `bytes` bytes at window address `addr` of CTA c, or nullptr (recorded) when outside the window
static uint8_t* window_ptr(Cta* c, uint32_t addr, size_t bytes, const char* what) {
  const uint32_t off = addr & 0xffffffu;
  if (off >= c->dyn_base && (size_t)off + bytes <= (size_t)c->dyn_base + c->dyn_bytes) return c->dyn + (off - c->dyn_base);
  if (off >= 16 && off < kDynWindowBase && bytes <= 8) {
    const size_t i = (off - 16) / 8;
    if (i < c->statics.size()) return (uint8_t*)c->statics[i] + (off & 7);
  }
  violation("%s: %s touches shared memory [0x%x, +%zu) outside the CTA's window [0x%x, +%zu) (CTA %u,%u)", c->gang->kernel, what, off,
            bytes, c->dyn_base, c->dyn_bytes, c->bid.x, c->bid.y);
  return nullptr;
}
uint32_t ld_shared_u32(uint32_t addr) {
  Cta* c = owner_of(addr, cur()->cta);
  uint8_t* p = c ? window_ptr(c, addr, 4, "ld.shared") : nullptr;
  uint32_t v = 0;
  if (p) memcpy(&v, p, 4);
  return v;
}
void st_shared_u32(uint32_t addr, uint32_t v) {
  Cta* c = owner_of(addr, cur()->cta);
  uint8_t* p = c ? window_ptr(c, addr, 4, "st.shared") : nullptr;
  if (p) memcpy(p, &v, 4);
  note_progress();
}

// ------------------------------------------------------------------------------------------------------------------
// mbarrier
constexpr uint64_t kMbarCookie = 0x6d62617272696572ull;    // written into the 8 bytes an initialised barrier occupies
static Mbar* mbar_at(Cta* c, uint32_t addr, const char* what) {
  const uint32_t off = addr & 0xffffffu;
  if (off & 7) { violation("%s: %s on a misaligned mbarrier address 0x%x", c->gang->kernel, what, off); return nullptr; }
  uint8_t* p = window_ptr(c, addr, 8, what);
  if (!p) return nullptr;
  auto it = c->mbars.find(off);
  if (it == c->mbars.end()) { violation("%s: %s on shared memory 0x%x that holds no initialised mbarrier (CTA %u,%u)", c->gang->kernel, what, off, c->bid.x, c->bid.y); return nullptr; }
  uint64_t cookie; memcpy(&cookie, p, 8);
  if (cookie != kMbarCookie) { violation("%s: the mbarrier at 0x%x was overwritten (CTA %u,%u)", c->gang->kernel, off, c->bid.x, c->bid.y); return nullptr; }
  return &it->second;
}
static void mbar_check_complete(Mbar* b) {
  if (b->pending == 0 && b->tx == 0) { b->phase ^= 1; b->pending = b->expected; }
  note_progress();
}
void mbar_init(uint32_t addr, uint32_t count) {
  Cta* c = cur()->cta;
  if ((addr >> 24) != 0) { violation("%s: mbarrier.init through a shared::cluster address", c->gang->kernel); return; }
  const uint32_t off = addr & 0xffffffu;
  uint8_t* p = (off & 7) ? nullptr : window_ptr(c, addr, 8, "mbarrier.init");
  if (!p || count == 0 || count > (1u << 20) - 1) { violation("%s: mbarrier.init(0x%x, %u) invalid", c->gang->kernel, off, count); return; }
  memcpy(p, &kMbarCookie, 8);
  Mbar b; b.expected = b.pending = count;
  c->mbars[off] = b;
  note_progress();
}
static void mbar_arrive_on(Cta* c, uint32_t addr, uint32_t tx_bytes, const char* what) {
  Mbar* b = mbar_at(c, addr, what);
  if (!b) return;
  b->tx += tx_bytes;
  if (b->pending == 0) { violation("%s: %s: more arrivals than the barrier at 0x%x expects in one phase", c->gang->kernel, what, addr & 0xffffffu); return; }
  b->pending--;
  mbar_check_complete(b);
}
static void mbar_complete_tx(Cta* c, uint32_t addr, uint32_t bytes, const char* what) {
  Mbar* b = mbar_at(c, addr, what);
  if (!b) return;
  b->tx -= bytes;
  mbar_check_complete(b);
}
void mbar_arrive(uint32_t addr, uint32_t tx_bytes) {
  Cta* c = owner_of(addr, cur()->cta);
  if (c) mbar_arrive_on(c, addr, tx_bytes, tx_bytes ? "mbarrier.arrive.expect_tx" : "mbarrier.arrive");
}
bool mbar_try_wait(uint32_t addr, uint32_t parity) {
  Cta* self = cur()->cta;
  if ((addr >> 24) != 0 && owner_of(addr, self) != self) { violation("%s: mbarrier.try_wait on another CTA's barrier", self->gang->kernel); return true; }
  for (int attempt = 0; attempt < 2; ++attempt) {
    Mbar* b = mbar_at(self, addr, "mbarrier.try_wait");
    if (!b) return true;                       // recorded; do not spin on it
    if (b->phase != (parity & 1)) { note_progress(); return true; }
    g_fiber->where = "mbarrier.try_wait"; g_fiber->where_arg = addr;
    if (attempt == 0) yield();                 // potentially blocking: gives the others one turn, then reports
  }
  return false;
}

// ------------------------------------------------------------------------------------------------------------------
// TMA.  The emulated cuTensorMapEncodeTiled stores this record in the 128 opaque bytes of a CUtensorMap.
struct EmuMap {
  uint64_t magic;
  const char* base;
  uint32_t rank, swizzle, elem;
  uint64_t dims[5], strides[4];
  uint32_t box[5];
};
static_assert(sizeof(EmuMap) <= sizeof(CUtensorMap), "the emulated tensor map must fit the opaque one");
constexpr uint64_t kMapMagic = 0x656d756d61703031ull;

static inline uint32_t swizzle_addr(uint32_t a, uint32_t mode) {
  if (mode == CU_TENSOR_MAP_SWIZZLE_128B) return a ^ (((a >> 7) & 7u) << 4);
  if (mode == CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B) return a ^ (((a >> 7) & 3u) << 5);
  return a;
}

void tma_load(const CUtensorMap* map, uint32_t dst, uint32_t bar, int c0, int c1, int c2, bool pair) {
  ThreadCtx* t = cur();
  Cta* c = t->cta;
  Gang* g = c->gang;
  EmuMap m; memcpy(&m, map, sizeof m);
  if (m.magic != kMapMagic || m.rank != 3) { violation("%s: TMA load through something that is not an encoded rank-3 tensor map", g->kernel); return; }
  if (pair && g->ctas.size() != 2) { violation("%s: cta_group::2 TMA load outside a CTA pair", g->kernel); return; }
  if (dst & 127u) { violation("%s: TMA destination 0x%x is not 128-byte aligned", g->kernel, dst); return; }
  if (m.swizzle != CU_TENSOR_MAP_SWIZZLE_NONE && (dst & 1023u) && g_cfg.verbose)
    fprintf(stderr, "[emu] note: swizzled TMA destination 0x%x is not 1024-byte aligned\n", dst);
  const size_t bytes = (size_t)m.box[0] * m.box[1] * m.box[2] * m.elem;
  Cta* bar_cta = owner_of(bar, c);
  if (!bar_cta) return;
  const long id = g_tma_count++;
  g_traffic[g->kernel][0] += (long)bytes;
  const int coord[3] = {c0, c1, c2};
  check_smem_write_issue(g, c, dst, dst + (uint32_t)bytes, "TMA load");
  asan_guard(c, dst, bytes, true);
  Touch touch; touch.smem_w.push_back(Range{c, dst, dst + (uint32_t)bytes});
  post(g, [=]() {
    asan_guard(c, dst, bytes, false);
    uint8_t* base = window_ptr(c, dst, bytes, "TMA load");
    if (base) {
      for (uint32_t i2 = 0; i2 < m.box[2]; ++i2)
        for (uint32_t i1 = 0; i1 < m.box[1]; ++i1) {
          const long long y = (long long)coord[1] + i1, z = (long long)coord[2] + i2;
          for (uint32_t i0 = 0; i0 < m.box[0]; ++i0) {
            const long long x = (long long)coord[0] + i0;
            float v = 0.f;                                             // out-of-bounds elements are filled with zeros
            if (x >= 0 && y >= 0 && z >= 0 && (uint64_t)x < m.dims[0] && (uint64_t)y < m.dims[1] && (uint64_t)z < m.dims[2]) {
              const char* src = m.base + (size_t)x * m.elem + (size_t)y * m.strides[0] + (size_t)z * m.strides[1];
              if (!in_device(src, m.elem)) { violation("%s: TMA reads outside the device allocation of its tensor", g->kernel); return; }
              memcpy(&v, src, 4);
            }
            const uint32_t lin = ((i2 * m.box[1] + i1) * m.box[0] + i0) * m.elem;
            const uint32_t a = swizzle_addr(dst + lin, m.swizzle);
            memcpy(base + (a - dst), &v, 4);
          }
        }
    }
    if (id == g_cfg.drop_tma) return;                                  // injected fault: the completion is lost
    mbar_complete_tx(bar_cta, bar, (uint32_t)bytes, "TMA complete_tx");
  }, std::move(touch));
}

// plain bulk copies
void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  Cta* c = cur()->cta;
  Gang* g = c->gang;
  if ((dst & 15u) || ((uintptr_t)src & 15u) || (bytes & 15u) || bytes == 0) { violation("%s: cp.async.bulk needs 16-byte aligned addresses and size (dst 0x%x, src %p, %u bytes)", g->kernel, dst, src, bytes); return; }
  if (!in_device(src, bytes)) { violation("%s: cp.async.bulk reads [%p, +%u) outside every device allocation", g->kernel, src, bytes); return; }
  const long id = g_tma_count++;
  g_traffic[g->kernel][0] += (long)bytes;
  check_smem_write_issue(g, c, dst, dst + bytes, "cp.async.bulk");
  asan_guard(c, dst, bytes, true);
  Touch touch; touch.smem_w.push_back(Range{c, dst, dst + bytes});
  // the copy engine may read its source any time between issue and completion: either extreme, by the schedule's seed
  std::shared_ptr<std::vector<uint8_t>> early;
  if (rnd(g) & 1) early = std::make_shared<std::vector<uint8_t>>((const uint8_t*)src, (const uint8_t*)src + bytes);
  post(g, [=]() {
    asan_guard(c, dst, bytes, false);
    uint8_t* p = window_ptr(c, dst, bytes, "cp.async.bulk (global -> shared)");
    if (p) memcpy(p, early ? early->data() : (const uint8_t*)src, bytes);
    if (id == g_cfg.drop_tma) return;
    mbar_complete_tx(c, bar, bytes, "cp.async.bulk complete_tx");
  }, std::move(touch));
}
void bulk_s2g(void* dst, uint32_t src, uint32_t bytes) {
  Cta* c = cur()->cta;
  Gang* g = c->gang;
  Fiber* f = g_fiber;
  if ((src & 15u) || ((uintptr_t)dst & 15u) || (bytes & 15u) || bytes == 0) { violation("%s: cp.async.bulk needs 16-byte aligned addresses and size (src 0x%x, dst %p, %u bytes)", g->kernel, src, dst, bytes); return; }
  if (!in_device(dst, bytes)) { violation("%s: cp.async.bulk writes [%p, +%u) outside every device allocation", g->kernel, dst, bytes); return; }
  f->bulk_pending++;
  post(g, [=]() {
    uint8_t* p = window_ptr(c, src, bytes, "cp.async.bulk (shared -> global)");
    if (p) memcpy(dst, p, bytes);
    f->bulk_pending--;
  });
}
void bulk_wait_read() {
  Fiber* f = g_fiber;
  while (f->bulk_pending > 0) yield();
  note_progress();
}

// ------------------------------------------------------------------------------------------------------------------
// tcgen05
void tmem_alloc(uint32_t dst_addr, uint32_t ncols, bool pair) {
  ThreadCtx* t = cur();
  Cta* c = t->cta;
  const int leader = __builtin_ctz(c->warps[t->warp].live);
  warp_barrier(0xffffffffu);                      // .sync.aligned: the whole warp executes it
  if (t->lane != leader) return;
  if (pair && c->gang->ctas.size() != 2) { violation("%s: cta_group::2 tcgen05.alloc outside a CTA pair", c->gang->kernel); return; }
  if (ncols < 32 || ncols > 512 || (ncols & (ncols - 1))) { violation("%s: tcgen05.alloc of %u columns (power of two in [32, 512] required)", c->gang->kernel, ncols); return; }
  if (c->tmem_allocated) { violation("%s: second tcgen05.alloc in one CTA (would block for ever with all 512 columns taken)", c->gang->kernel); return; }
  c->tmem_allocated = true; c->tmem_cols = ncols;
  uint8_t* p = window_ptr(c, dst_addr, 4, "tcgen05.alloc result");
  const uint32_t base = 0;
  if (p) memcpy(p, &base, 4);
  note_progress();
}
void tmem_dealloc(uint32_t taddr, uint32_t ncols, bool pair) {
  ThreadCtx* t = cur();
  Cta* c = t->cta;
  (void)pair;
  const int leader = __builtin_ctz(c->warps[t->warp].live);
  warp_barrier(0xffffffffu);
  if (t->lane != leader) return;
  if (!c->tmem_allocated || taddr != 0 || ncols != c->tmem_cols) { violation("%s: tcgen05.dealloc(0x%x, %u) does not match the allocation (%s, %u columns) in CTA (%u,%u)", c->gang->kernel, taddr, ncols, c->tmem_allocated ? "allocated" : "nothing allocated", c->tmem_cols, c->bid.x, c->bid.y); return; }
  if (!c->gang->pipe.empty()) violation("%s: tcgen05.dealloc while MMAs or commits of the CTA are still in flight", c->gang->kernel);
  c->tmem_allocated = false;
  note_progress();
}
static uint32_t* tmem_cell(Cta* c, uint32_t lane, uint32_t col, const char* what) {
  if (!c->tmem_allocated || lane >= (uint32_t)kTmemLanes || col >= c->tmem_cols) {
    violation("%s: %s touches TMEM lane %u column %u outside the allocation of %u columns", c->gang->kernel, what, lane, col, c->tmem_allocated ? c->tmem_cols : 0u);
    return nullptr;
  }
  return &c->tmem[(size_t)lane * kTmemCols + col];
}
void tmem_ld32(uint32_t taddr, uint32_t* v) {
  ThreadCtx* t = cur();
  Cta* c = t->cta;
  warp_barrier(0xffffffffu);
  const uint32_t lane0 = taddr >> 16, col = taddr & 0xffffu;
  check_tmem_thread_access(c->gang, c, col, col + 32, false, "tcgen05.ld");
  if (lane0 != (uint32_t)(t->warp & 3) * 32u) violation("%s: tcgen05.ld from lanes %u.. by warp %d (a warp may only touch lane quadrant warp %% 4)", c->gang->kernel, lane0, t->warp);
  for (uint32_t j = 0; j < 32; ++j) {
    uint32_t* p = tmem_cell(c, lane0 + (uint32_t)t->lane, col + j, "tcgen05.ld");
    v[j] = p ? *p : 0x7fc00000u;
  }
}
void tmem_st32(uint32_t taddr, const uint32_t* v) {
  ThreadCtx* t = cur();
  Cta* c = t->cta;
  warp_barrier(0xffffffffu);
  const uint32_t lane0 = taddr >> 16, col = taddr & 0xffffu;
  check_tmem_thread_access(c->gang, c, col, col + 32, true, "tcgen05.st");
  if (lane0 != (uint32_t)(t->warp & 3) * 32u) violation("%s: tcgen05.st to lanes %u.. by warp %d (a warp may only touch lane quadrant warp %% 4)", c->gang->kernel, lane0, t->warp);
  for (uint32_t j = 0; j < 32; ++j) {
    uint32_t* p = tmem_cell(c, lane0 + (uint32_t)t->lane, col + j, "tcgen05.st");
    if (p) *p = v[j];
  }
  note_progress();
}

void tc_commit(uint32_t bar, bool pair) {
  Cta* c = cur()->cta;
  Gang* g = c->gang;
  if (pair && g->ctas.size() != 2) { violation("%s: cta_group::2 tcgen05.commit outside a CTA pair", g->kernel); return; }
  const long id = g_commit_count++;
  post_pipe(g, [=]() {
    if (id == g_cfg.drop_commit) return;                               // injected fault
    if (pair) { for (auto& cc : g->ctas) mbar_arrive_on(cc.get(), bar & 0xffffffu, 0, "tcgen05.commit"); }   // multicast to both CTAs, same offset
    else { Cta* o = owner_of(bar, c); if (o) mbar_arrive_on(o, bar, 0, "tcgen05.commit"); }
  });
}

// operand gather.  desc: start address (16 B units, 14 bits) | LBO << 16 | SBO << 32 | version << 46 | layout << 61
struct Desc { uint32_t start, lbo, sbo, layout, version, base_offset; };
static Desc decode_desc(uint64_t d) {
  Desc r;
  r.start = (uint32_t)(d & 0x3fff) << 4;
  r.lbo = (uint32_t)((d >> 16) & 0x3fff) << 4;
  r.sbo = (uint32_t)((d >> 32) & 0x3fff) << 4;
  r.version = (uint32_t)((d >> 46) & 3);
  r.base_offset = (uint32_t)((d >> 49) & 7);
  r.layout = (uint32_t)((d >> 61) & 7);
  return r;
}
static inline float tf32_of(uint32_t bits) { bits &= 0xffffe000u; float f; memcpy(&f, &bits, 4); return f; }   // the tensor core ignores the low 13 bits

// rows x 8 tf32 operand from shared memory into out[rows][8]
static bool gather_smem(Cta* c, uint64_t desc, bool mn_major, int rows, float* out, const char* what) {
  const Desc d = decode_desc(desc);
  if (d.version != 1) { violation("%s: %s descriptor version %u (sm_100 needs 1)", c->gang->kernel, what, d.version); return false; }
  if (d.base_offset != 0) { violation("%s: %s descriptor base offset %u is not modelled", c->gang->kernel, what, d.base_offset); return false; }
  if (!mn_major) {
    if (d.layout != 2) { violation("%s: %s K-major tf32 operand with layout type %u (only SWIZZLE_128B = 2 is modelled)", c->gang->kernel, what, d.layout); return false; }
    for (int r = 0; r < rows; ++r)
      for (int k = 0; k < 8; ++k) {
        const uint32_t a = d.start + (uint32_t)(r >> 3) * d.sbo + (uint32_t)(r & 7) * 128u + (uint32_t)k * 4u;
        const uint32_t s = a ^ (((a >> 7) & 7u) << 4);
        uint8_t* p = window_ptr(c, s, 4, what);
        if (!p) return false;
        uint32_t bits; memcpy(&bits, p, 4);
        out[r * 8 + k] = tf32_of(bits);
      }
  } else {
    if (d.layout != 1) { violation("%s: %s MN-major tf32 operand with layout type %u (tf32 has SWIZZLE_128B_BASE32B = 1 only)", c->gang->kernel, what, d.layout); return false; }
    for (int r = 0; r < rows; ++r)
      for (int k = 0; k < 8; ++k) {
        const uint32_t a = d.start + (uint32_t)(r >> 5) * d.lbo + (uint32_t)(k >> 2) * d.sbo + (uint32_t)(k & 3) * 128u + (uint32_t)(r & 31) * 4u;
        const uint32_t s = a ^ (((a >> 7) & 3u) << 5);
        uint8_t* p = window_ptr(c, s, 4, what);
        if (!p) return false;
        uint32_t bits; memcpy(&bits, p, 4);
        out[r * 8 + k] = tf32_of(bits);
      }
  }
  return true;
}
static inline float trunc_to_f32(double x) {        // the tensor core's accumulate does not round to nearest: it truncates
  float f = (float)x;
  if (fabs((double)f) > fabs(x)) f = nextafterf(f, 0.f);
  return f;
}

void tc_mma(uint32_t d_tmem, bool a_in_tmem, uint32_t a_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc, bool pair) {
  Cta* c = cur()->cta;
  Gang* g = c->gang;
  g_mma_count++;
  // what this MMA will touch (decoded the way the execution below decodes it), checked against the copies in flight
  Touch touch;
  {
    const int N = (int)((idesc >> 17) & 0x3f) << 3, a_mn = (int)(idesc >> 15) & 1, b_mn = (int)(idesc >> 16) & 1;
    const int ncta = pair ? 2 : 1;
    {
      std::array<long, 3>& t = g_traffic[g->kernel];
      t[1] += (long)ncta * ((N / ncta) * 32 + (a_in_tmem ? 0 : 128 * 32));      // rows x 8 tf32 words per operand and CTA
      t[2] += (long)ncta * (N / 2);
    }
    auto operand = [&](const Cta* cc, uint64_t desc, bool mn, int rows) {
      const uint32_t start = (uint32_t)(desc & 0x3fff) << 4, lbo = (uint32_t)((desc >> 16) & 0x3fff) << 4, sbo = (uint32_t)((desc >> 32) & 0x3fff) << 4;
      if (!mn) touch.smem_r.push_back(Range{cc, start & ~127u, (start & ~127u) + (uint32_t)((rows + 7) / 8 - 1) * sbo + 1024u});
      else for (int grp = 0; grp < (rows + 31) / 32; ++grp) touch.smem_r.push_back(Range{cc, start + (uint32_t)grp * lbo, start + (uint32_t)grp * lbo + sbo + 512u});
    };
    for (int h = 0; h < ncta && (size_t)(pair ? h : c->rank) < g->ctas.size(); ++h) {
      const Cta* cc = g->ctas[(size_t)(pair ? h : c->rank)].get();
      operand(cc, b_desc, b_mn != 0, N / ncta);
      if (a_in_tmem) touch.tmem_r.push_back(Cols{cc, a_tmem & 0xffffu, (a_tmem & 0xffffu) + 8u});
      else operand(cc, a_desc, a_mn != 0, 128);
      touch.tmem_w.push_back(Cols{cc, d_tmem & 0xffffu, (d_tmem & 0xffffu) + (uint32_t)N});
    }
    for (const Range& r : touch.smem_r) check_smem_read_issue(g, r.cta, r.lo, r.hi, "tcgen05.mma");
  }
  post_pipe(g, [=]() {
    const int M = (int)((idesc >> 24) & 0x1f) << 4, N = (int)((idesc >> 17) & 0x3f) << 3;
    const int a_mn = (int)(idesc >> 15) & 1, b_mn = (int)(idesc >> 16) & 1;
    const int dfmt = (int)(idesc >> 4) & 3, afmt = (int)(idesc >> 7) & 7, bfmt = (int)(idesc >> 10) & 7;
    if (dfmt != 1 || afmt != 2 || bfmt != 2) { violation("%s: tcgen05.mma kind::tf32 with formats D %d A %d B %d (need 1, 2, 2)", g->kernel, dfmt, afmt, bfmt); return; }
    if (idesc & ((1u << 13) | (1u << 14) | 0xfu | (1u << 6))) { violation("%s: instruction descriptor 0x%x sets negate / sparsity / saturate bits", g->kernel, idesc); return; }
    const int ncta = pair ? 2 : 1;
    if (pair && (g->ctas.size() != 2 || c->rank != 0)) { violation("%s: cta_group::2 MMA must be issued by the leader of a CTA pair", g->kernel); return; }
    if (M != 128 * ncta) { violation("%s: tcgen05.mma M = %d with cta_group::%d", g->kernel, M, ncta); return; }
    if (N < 16 || N > 256 || (N % 16)) { violation("%s: tcgen05.mma N = %d (multiple of 16 in [16, 256] required for M = 128 per CTA)", g->kernel, N); return; }
    if ((d_tmem >> 16) != 0) { violation("%s: accumulator address 0x%x does not start at lane 0", g->kernel, d_tmem); return; }
    if (a_in_tmem && a_mn) { violation("%s: A from TMEM cannot be MN-major", g->kernel); return; }
    const uint32_t dcol = d_tmem & 0xffffu;
    // B: N rows; with a CTA pair each CTA's shared memory holds N / 2 of them at the same offset
    std::vector<float> B((size_t)N * 8), A((size_t)128 * 8);
    const int nb = N / ncta;
    for (int h = 0; h < ncta; ++h)
      if (!gather_smem(g->ctas[(size_t)(pair ? h : c->rank)].get(), b_desc, b_mn != 0, nb, B.data() + (size_t)h * nb * 8, "tcgen05.mma B operand")) return;
    for (int h = 0; h < ncta; ++h) {
      Cta* cc = g->ctas[(size_t)(pair ? h : c->rank)].get();
      if (a_in_tmem) {
        if ((a_tmem >> 16) != 0) { violation("%s: A operand TMEM address 0x%x does not start at lane 0", g->kernel, a_tmem); return; }
        for (int r = 0; r < 128; ++r)
          for (int k = 0; k < 8; ++k) {
            uint32_t* p = tmem_cell(cc, (uint32_t)r, (a_tmem & 0xffffu) + (uint32_t)k, "tcgen05.mma A operand");
            if (!p) return;
            A[(size_t)r * 8 + k] = tf32_of(*p);
          }
      } else if (!gather_smem(cc, a_desc, a_mn != 0, 128, A.data(), "tcgen05.mma A operand")) return;
      if (!tmem_cell(cc, 0, dcol, "tcgen05.mma accumulator") || !tmem_cell(cc, 127, dcol + (uint32_t)N - 1, "tcgen05.mma accumulator")) return;
      for (int r = 0; r < 128; ++r) {
        const float* ar = &A[(size_t)r * 8];
        uint32_t* drow = &cc->tmem[(size_t)r * kTmemCols + dcol];
        for (int n = 0; n < N; ++n) {
          const float* br = &B[(size_t)n * 8];
          double s = 0.0;
          for (int k = 0; k < 8; ++k) s += (double)ar[k] * (double)br[k];
          float dv = 0.f;
          if (acc) memcpy(&dv, &drow[n], 4);
          const float nv = trunc_to_f32((double)dv + s);
          memcpy(&drow[n], &nv, 4);
        }
      }
    }
  }, std::move(touch));
}

// ------------------------------------------------------------------------------------------------------------------
// launches
struct Graph;
struct Stream { Graph* capture = nullptr; };
struct Node { std::string name; LaunchCfg cfg; const void* fn; std::function<void()> body; };
struct CondHandle { unsigned value = 0, dflt = 0; bool assign_default = false; };
struct Graph {
  std::vector<Node> nodes;               // kernel nodes in capture order
  int cond_handle = -1;                  // >= 0: this graph is a single WHILE node over `body`
  std::unique_ptr<Graph> body;
};
static std::vector<std::unique_ptr<CondHandle>> g_handles;
static std::map<const void*, int> g_smem_cap;

static void execute(const LaunchCfg& cfg, const char* name, const std::function<void()>& body) {
  g_kernel_runs[name]++;
  if (g_sticky != cudaSuccess) return;
  struct Timer {
    const char* n; timespec t0;
    explicit Timer(const char* nn) : n(nn) { clock_gettime(CLOCK_MONOTONIC, &t0); }
    ~Timer() { timespec t1; clock_gettime(CLOCK_MONOTONIC, &t1); g_kernel_secs[n] += (double)(t1.tv_sec - t0.tv_sec) + 1e-9 * (double)(t1.tv_nsec - t0.tv_nsec); }
  } timer(name);
  const int nthreads = (int)(cfg.block.x * cfg.block.y * cfg.block.z);
  const int cl = cfg.cluster_x;
  static uint64_t launch_seq = 0;
  ++launch_seq;
  for (unsigned bz = 0; bz < cfg.grid.z; ++bz)
    for (unsigned by = 0; by < cfg.grid.y; ++by)
      for (unsigned bx0 = 0; bx0 < cfg.grid.x; bx0 += (unsigned)cl) {
        Gang g;
        g.body = &body; g.kernel = name;
        g.rng = (g_cfg.seed * 0x9E3779B97F4A7C15ull) ^ (launch_seq << 20) ^ ((uint64_t)by << 10) ^ bx0 ^ 0x5851F42D4C957F2Dull;
        if (!g.rng) g.rng = 1;
        for (int r = 0; r < cl; ++r) {
          auto c = std::make_unique<Cta>();
          c->rank = r; c->bid = make_uint3(bx0 + (unsigned)r, by, bz);
          c->dyn_bytes = cfg.smem;
          c->dyn_base = kDynWindowBase + (uint32_t)g_cfg.dyn_misalign;
          void* region = nullptr;
          if (posix_memalign(&region, kWindowBytes, kWindowBytes)) abort();
          c->region = (uint8_t*)region;
          c->dyn = c->region + c->dyn_base;                  // a kernel that aligns the generic pointer aligns the window address
          memset(c->region, 0xCD, kWindowBytes);             // shared memory is not zero at kernel start
#if EMU_ASAN
          // memcheck for the kernels' own (generic) loads and stores: only the launched bytes are addressable
          __asan_poison_memory_region(c->region, kWindowBytes);
          __asan_unpoison_memory_region(c->dyn, cfg.smem);
#endif
          c->tmem.assign((size_t)kTmemLanes * kTmemCols, 0x7fc00000u);
          c->nthreads = c->live = nthreads;
          c->warps.resize((size_t)(nthreads + 31) / 32);
          c->gang = &g;
          for (int t = 0; t < nthreads; ++t) {
            auto f = std::make_unique<Fiber>();
            f->gang = &g;
            ThreadCtx& x = f->ctx;
            x.lin = t;
            x.tid = make_uint3((unsigned)t % cfg.block.x, ((unsigned)t / cfg.block.x) % cfg.block.y, (unsigned)t / (cfg.block.x * cfg.block.y));
            x.bid = c->bid; x.bdim = cfg.block; x.gdim = cfg.grid;
            x.warp = t >> 5; x.lane = t & 31; x.cta = c.get();
            c->warps[(size_t)x.warp].live |= 1u << x.lane;
            make_fiber(f.get());
            g.fibers.push_back(std::move(f));
          }
          g.live += nthreads;
          g.ctas.push_back(std::move(c));
        }
        run_gang(&g);
        for (auto& c : g.ctas) {
#if EMU_ASAN
          __asan_unpoison_memory_region(c->region, kWindowBytes);
#endif
          free(c->region);
        }
        if (g.hung) { g_sticky = cudaErrorLaunchFailure; return; }
      }
}

void submit(const LaunchCfg& cfg, const char* name, const void* fn, std::function<void()> body) {
  const unsigned nthreads = cfg.block.x * cfg.block.y * cfg.block.z;
  auto it = g_smem_cap.find(fn);
  const size_t cap = it == g_smem_cap.end() ? 48u * 1024u : (size_t)it->second;
  if (!cfg.grid.x || !cfg.grid.y || !cfg.grid.z || !nthreads || nthreads > 1024 || cfg.grid.y > 65535 || cfg.grid.z > 65535 ||
      (cfg.grid.x % (unsigned)cfg.cluster_x)) { g_last_error = cudaErrorInvalidConfiguration; return; }
  if (cfg.smem > cap) { g_last_error = cudaErrorInvalidValue; return; }
  Stream* st = reinterpret_cast<Stream*>(cfg.stream);
  const bool capturing = st && st->capture;
  g_launches.push_back(LaunchRec{name, cfg.grid, cfg.block, cfg.smem, capturing ? 1 : 0});
  if (capturing) { st->capture->nodes.push_back(Node{name, cfg, fn, std::move(body)}); return; }
  execute(cfg, name, body);
}

}  // namespace emu

// device-side API used by k_loop_cond
void cudaGraphSetConditional(cudaGraphConditionalHandle h, unsigned value) {
  if (h == 0 || h > emu::g_handles.size()) { emu::violation("cudaGraphSetConditional on an unknown handle"); return; }
  emu::g_handles[(size_t)h - 1]->value = value;
}

// ------------------------------------------------------------------------------------------------------------------
// the CUDA runtime API, as far as libgmco uses it
using namespace emu;
extern "C" {

cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
cudaError_t cudaDeviceGetAttribute(int* v, enum cudaDeviceAttr attr, int) {
  if (attr == cudaDevAttrComputeCapabilityMajor) *v = 10;
  else if (attr == cudaDevAttrMultiProcessorCount) *v = g_cfg.sm_count;
  else *v = 0;
  return cudaSuccess;
}
cudaError_t cudaGetLastError(void) { cudaError_t e = g_sticky != cudaSuccess ? g_sticky : g_last_error; g_last_error = cudaSuccess; return e; }
cudaError_t cudaPeekAtLastError(void) { return g_sticky != cudaSuccess ? g_sticky : g_last_error; }
const char* cudaGetErrorString(cudaError_t e) {
  return e == cudaSuccess ? "no error" : e == cudaErrorInvalidConfiguration ? "invalid configuration argument"
       : e == cudaErrorLaunchFailure ? "unspecified launch failure (emulated: the kernel hung)" : "emulated runtime error";
}
cudaError_t cudaDeviceGetDefaultMemPool(cudaMemPool_t* p, int) { static int pool; *p = (cudaMemPool_t)&pool; return cudaSuccess; }
cudaError_t cudaMemPoolSetAttribute(cudaMemPool_t, enum cudaMemPoolAttr, void*) { return cudaSuccess; }
cudaError_t cudaFuncSetAttribute(const void* func, enum cudaFuncAttribute attr, int value) {
  if (attr != cudaFuncAttributeMaxDynamicSharedMemorySize || value < 0 || value > 227 * 1024) return cudaErrorInvalidValue;
  g_smem_cap[func] = value;
  return cudaSuccess;
}

cudaError_t cudaMallocAsync(void** p, size_t n, cudaStream_t) {
  void* q = nullptr;
  if (posix_memalign(&q, 512, n ? n : 1)) return cudaErrorMemoryAllocation;
  memset(q, 0xFF, n);                       // fresh device memory is not zero: NaN for floats, -1 for ints
  g_allocs.push_back(Alloc{(char*)q, n});
  *p = q;
  return cudaSuccess;
}
cudaError_t cudaFreeAsync(void* p, cudaStream_t) {
  for (Alloc& a : g_allocs)
    if (a.p == p) { free(p); a.p = nullptr; a.n = 0; return cudaSuccess; }
  violation("cudaFreeAsync of %p, which is not a live allocation", p);
  return cudaErrorInvalidValue;
}
cudaError_t cudaPointerGetAttributes(struct cudaPointerAttributes* a, const void* p) {
  memset(a, 0, sizeof *a);
  a->type = find_alloc(p) ? cudaMemoryTypeDevice : cudaMemoryTypeUnregistered;
  return cudaSuccess;
}
static void check_range(const char* what, const void* p, size_t n) {
  const Alloc* a = find_alloc(p);
  if (a && (const char*)p + n > a->p + a->n) violation("%s [%p, +%zu) runs past its allocation", what, p, n);
}
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, enum cudaMemcpyKind, cudaStream_t) {
  check_range("cudaMemcpy destination", d, n); check_range("cudaMemcpy source", s, n);
  if (d && s && n) memmove(d, s, n);
  return g_sticky;
}
cudaError_t cudaMemcpy(void* d, const void* s, size_t n, enum cudaMemcpyKind k) { return cudaMemcpyAsync(d, s, n, k, nullptr); }
cudaError_t cudaMemcpy2DAsync(void* d, size_t dp, const void* s, size_t sp, size_t w, size_t h, enum cudaMemcpyKind, cudaStream_t) {
  if (w > dp || w > sp) return cudaErrorInvalidValue;
  if (h) { check_range("cudaMemcpy2D destination", d, (h - 1) * dp + w); check_range("cudaMemcpy2D source", s, (h - 1) * sp + w); }
  for (size_t r = 0; r < h; ++r) memmove((char*)d + r * dp, (const char*)s + r * sp, w);
  return g_sticky;
}
cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t) {
  if (!find_alloc(d)) { violation("cudaMemset of %p, which is not device memory", d); return cudaErrorInvalidValue; }
  check_range("cudaMemset", d, n);
  memset(d, v, n);
  return cudaSuccess;
}

cudaError_t cudaStreamSynchronize(cudaStream_t) { return g_sticky; }
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* st, unsigned) { *st = reinterpret_cast<cudaStream_t>(new Stream()); return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t st) { delete reinterpret_cast<Stream*>(st); return cudaSuccess; }
cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = (cudaEvent_t)malloc(8); return cudaSuccess; }
cudaError_t cudaEventDestroy(cudaEvent_t e) { free(e); return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t) { return e ? cudaSuccess : cudaErrorInvalidValue; }
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) { if (!a || !b) return cudaErrorInvalidValue; *ms = 0.01f; return cudaSuccess; }

// graphs: a WHILE conditional node whose body is captured from a stream
cudaError_t cudaGraphCreate(cudaGraph_t* g, unsigned) { *g = reinterpret_cast<cudaGraph_t>(new Graph()); return cudaSuccess; }
cudaError_t cudaGraphDestroy(cudaGraph_t g) { delete reinterpret_cast<Graph*>(g); return cudaSuccess; }
cudaError_t cudaGraphConditionalHandleCreate(cudaGraphConditionalHandle* h, cudaGraph_t, unsigned dflt, unsigned flags) {
  auto c = std::make_unique<CondHandle>();
  c->dflt = dflt; c->assign_default = (flags & cudaGraphCondAssignDefault) != 0; c->value = dflt;
  g_handles.push_back(std::move(c));
  *h = (cudaGraphConditionalHandle)g_handles.size();
  return cudaSuccess;
}
cudaError_t cudaGraphAddNode(cudaGraphNode_t* node, cudaGraph_t graph, const cudaGraphNode_t*, size_t ndeps, struct cudaGraphNodeParams* p) {
  Graph* g = reinterpret_cast<Graph*>(graph);
  if (!g || ndeps || p->type != cudaGraphNodeTypeConditional || p->conditional.type != cudaGraphCondTypeWhile || p->conditional.size != 1 ||
      g->cond_handle >= 0 || p->conditional.handle == 0 || p->conditional.handle > g_handles.size())
    return cudaErrorInvalidValue;
  g->cond_handle = (int)p->conditional.handle - 1;
  g->body = std::make_unique<Graph>();
  static cudaGraph_t out[1];
  out[0] = reinterpret_cast<cudaGraph_t>(g->body.get());
  p->conditional.phGraph_out = out;
  *node = reinterpret_cast<cudaGraphNode_t>(g->body.get());
  return cudaSuccess;
}
cudaError_t cudaStreamBeginCaptureToGraph(cudaStream_t stream, cudaGraph_t graph, const cudaGraphNode_t*, const cudaGraphEdgeData*, size_t, enum cudaStreamCaptureMode) {
  Stream* st = reinterpret_cast<Stream*>(stream);
  if (!st || !graph || st->capture) return cudaErrorInvalidValue;     // the legacy stream cannot capture
  st->capture = reinterpret_cast<Graph*>(graph);
  return cudaSuccess;
}
cudaError_t cudaStreamEndCapture(cudaStream_t stream, cudaGraph_t* out) {
  Stream* st = reinterpret_cast<Stream*>(stream);
  if (!st || !st->capture) return cudaErrorInvalidValue;
  if (out) *out = nullptr;
  st->capture = nullptr;
  return cudaSuccess;
}
cudaError_t cudaGraphInstantiate(cudaGraphExec_t* e, cudaGraph_t g, unsigned long long) {
  if (!g) return cudaErrorInvalidValue;
  *e = reinterpret_cast<cudaGraphExec_t>(g);                           // the "executable" is the graph itself
  return cudaSuccess;
}
cudaError_t cudaGraphExecDestroy(cudaGraphExec_t) { return cudaSuccess; }
cudaError_t cudaGraphLaunch(cudaGraphExec_t e, cudaStream_t) {
  Graph* g = reinterpret_cast<Graph*>(e);
  if (!g) return cudaErrorInvalidValue;
  for (const Node& n : g->nodes) execute(n.cfg, n.name.c_str(), n.body);
  if (g->cond_handle >= 0) {
    CondHandle* h = g_handles[(size_t)g->cond_handle].get();
    if (h->assign_default) h->value = h->dflt;
    long guard = 0;
    while (h->value && g_sticky == cudaSuccess) {
      for (const Node& n : g->body->nodes) execute(n.cfg, n.name.c_str(), n.body);
      if (++guard > 10000000) { violation("conditional WHILE node did not terminate"); break; }
    }
  }
  return g_sticky;
}

// driver entry point: cuTensorMapEncodeTiled
static CUresult emu_encode_tiled(CUtensorMap* map, CUtensorMapDataType dtype, cuuint32_t rank, void* addr, const cuuint64_t* dims,
                                 const cuuint64_t* strides, const cuuint32_t* box, const cuuint32_t* estr, CUtensorMapInterleave interleave,
                                 CUtensorMapSwizzle swizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill oob) {
  if (!map || !addr || rank < 1 || rank > 5 || ((uintptr_t)addr & 15) || dtype != CU_TENSOR_MAP_DATA_TYPE_FLOAT32 ||
      interleave != CU_TENSOR_MAP_INTERLEAVE_NONE || oob != CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE)
    return CUDA_ERROR_INVALID_VALUE;
  if (!find_alloc(addr)) { violation("tensor map over %p, which is not device memory", addr); return CUDA_ERROR_INVALID_VALUE; }
  EmuMap m{};
  m.magic = kMapMagic; m.base = (const char*)addr; m.rank = rank; m.swizzle = (uint32_t)swizzle; m.elem = 4;
  for (unsigned i = 0; i < rank; ++i) {
    if (!dims[i] || dims[i] > (1ull << 32) || !box[i] || box[i] > 256 || estr[i] != 1) return CUDA_ERROR_INVALID_VALUE;
    if (i + 1 < rank && ((strides[i] & 15) || strides[i] >= (1ull << 40))) return CUDA_ERROR_INVALID_VALUE;
    m.dims[i] = dims[i]; m.box[i] = box[i];
    if (i + 1 < rank) m.strides[i] = strides[i];
  }
  const uint64_t inner = (uint64_t)box[0] * 4;
  if (swizzle == CU_TENSOR_MAP_SWIZZLE_128B || swizzle == CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B) { if (inner > 128) return CUDA_ERROR_INVALID_VALUE; }
  else if (swizzle != CU_TENSOR_MAP_SWIZZLE_NONE) return CUDA_ERROR_INVALID_VALUE;
  uint64_t far = dims[0] * 4;
  for (unsigned i = 1; i < rank; ++i) far += (dims[i] - 1) * strides[i - 1];
  if (!in_device(addr, far)) { violation("tensor map extent [%p, +%llu) runs past its allocation", addr, (unsigned long long)far); return CUDA_ERROR_INVALID_VALUE; }
  memset(map, 0, sizeof *map);
  memcpy(map, &m, sizeof m);
  return CUDA_SUCCESS;
}
cudaError_t cudaGetDriverEntryPoint(const char* name, void** fn, unsigned long long, enum cudaDriverEntryPointQueryResult* status) {
  if (strcmp(name, "cuTensorMapEncodeTiled")) { *fn = nullptr; if (status) *status = cudaDriverEntryPointSymbolNotFound; return cudaErrorInvalidValue; }
  *fn = (void*)emu_encode_tiled;
  if (status) *status = cudaDriverEntryPointSuccess;
  return cudaSuccess;
}

// ---- test hooks (ctypes) ----
#pragma GCC visibility push(default)
int emu_violations(void) { return g_violations; }
const char* emu_violation_message(void) { return g_violation_msg; }
void emu_clear(void) { g_traffic.clear(); g_violations = 0; g_violation_msg[0] = 0; g_launches.clear(); g_kernel_runs.clear(); g_kernel_secs.clear(); g_sticky = cudaSuccess; g_last_error = cudaSuccess; g_hangs = 0; }
int emu_live_allocations(void) { int n = 0; for (const Alloc& a : g_allocs) n += a.p != nullptr; return n; }
long emu_traffic(const char* kernel, int what) {     // what: 0 bytes landed, 1 bytes read by MMA operands, 2 tensor-pipe cycles x SMs
  auto it = g_traffic.find(kernel);
  return it == g_traffic.end() || what < 0 || what > 2 ? 0 : it->second[(size_t)what];
}
long emu_counter(const char* what) {
  const std::string w(what);
  if (w == "tma") return g_tma_count;
  if (w == "commit") return g_commit_count;
  if (w == "mma") return g_mma_count;
  if (w == "hangs") return g_hangs;
  if (w == "launches") return (long)g_launches.size();
  if (w == "executed") { long n = 0; for (const auto& kv : g_kernel_runs) n += kv.second; return n; }   // kernels run, graph replays included
  auto it = g_kernel_runs.find(w);
  long n = 0;
  for (const auto& kv : g_kernel_runs) if (kv.first.find(w) != std::string::npos) n += kv.second;
  return it != g_kernel_runs.end() ? it->second : n;
}
int emu_set(const char* key, long v) {
  const std::string k(key);
  if (k == "seed") g_cfg.seed = (uint64_t)v;
  else if (k == "max_delay") g_cfg.max_delay = (int)v;
  else if (k == "mma_delay") g_cfg.mma_delay = (int)v;
  else if (k == "dyn_misalign") g_cfg.dyn_misalign = (int)v;
  else if (k == "sm_count") g_cfg.sm_count = (int)v;
  else if (k == "drop_tma") g_cfg.drop_tma = v < 0 ? -1 : g_tma_count + v;
  else if (k == "drop_commit") g_cfg.drop_commit = v < 0 ? -1 : g_commit_count + v;
  else if (k == "shuffle") g_cfg.shuffle = (int)v;
  else if (k == "starve_mask") g_cfg.starve_mask = (unsigned)v;
  else if (k == "starve_period") g_cfg.starve_period = (int)v;
  else if (k == "verbose") g_cfg.verbose = (int)v;
  else return -1;
  return 0;
}
void emu_print_times(void) {
  for (const auto& kv : g_kernel_secs) fprintf(stderr, "[emu] %8.3f s  %6ld x  %s\n", kv.second, g_kernel_runs[kv.first], kv.first.c_str());
}
int emu_launch(int i, char* name, int cap, unsigned* dims, unsigned long long* smem, int* captured) {
  if (i < 0 || (size_t)i >= g_launches.size()) return -1;
  const LaunchRec& r = g_launches[(size_t)i];
  snprintf(name, (size_t)cap, "%s", r.name.c_str());
  dims[0] = r.grid.x; dims[1] = r.grid.y; dims[2] = r.grid.z; dims[3] = r.block.x; dims[4] = r.block.y; dims[5] = r.block.z;
  *smem = r.smem; *captured = r.captured;
  return 0;
}
#pragma GCC visibility pop

}  // extern "C"
