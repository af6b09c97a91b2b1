// emu_core.h -- TEST INFRASTRUCTURE ONLY: a CPU-side execution model of CUDA's SIMT programming model.
//
// tests/emu/ compiles the product's kernel SOURCE (paper_1904_01567_b200/csrc/*.cu) with g++ and runs it on the host
// so that the code paths of libgmco can be executed, bounds-checked and compared with the oracle on a machine that
// has no GPU.  It is not a fallback of the product: nothing under paper_1904_01567_b200/ includes, links or loads it,
// and the library it builds (tests/emu/_build/libgmco_emu.so) is only ever opened by tests/test_emu_*.py.
//
// Model: every CUDA thread of a CTA is a fiber (own stack, cooperative switching); a CTA (or, for clusters, the CTAs
// of one cluster) runs to completion before the next one starts.  __syncthreads, warp shuffles / votes, mbarriers,
// cluster barriers block by yielding.  Asynchronous hardware units (TMA, the tcgen05 tensor pipe, bulk copies) are
// modelled by a queue of operations that complete some scheduler ticks after they were issued (emu_ptx.h,
// emu_runtime.cc), so that a kernel which reads a buffer before its barrier said so reads stale data here as well.
#pragma once

#include <cuda_runtime.h>
#include <cuda.h>

#include <math.h>
#include <stdint.h>
#include <string.h>

#include <algorithm>
#include <functional>
#include <tuple>
#include <type_traits>
#include <utility>

// ---- CUDA decorations mean nothing to the host compiler ----
#undef __global__
#undef __device__
#undef __host__
#undef __shared__
#undef __forceinline__
#undef __launch_bounds__
#undef __align__
#undef __grid_constant__
#undef __cluster_dims__
#define __global__
#define __device__
#define __host__
#define __shared__ static thread_local
#define __forceinline__ inline __attribute__((always_inline))
#define __launch_bounds__(...)
#define __align__(n) __attribute__((aligned(n)))
#define __grid_constant__
#define __cluster_dims__(...)

namespace emu {

struct Cta;

// what a CUDA thread knows about itself
struct ThreadCtx {
  uint3 tid, bid;
  dim3 bdim, gdim;
  int lin;          // linear thread index in the CTA
  int warp, lane;
  Cta* cta;
};
extern thread_local ThreadCtx* g_cur;
inline ThreadCtx* cur() { return g_cur; }

void yield();                                   // let the other fibers run
void cta_barrier();                             // __syncthreads
void warp_barrier(unsigned mask);               // __syncwarp and the convergence point of every *.sync warp operation
void warp_exchange(unsigned mask, const void* in, void* out, int bytes, int src_lane);
unsigned warp_ballot(unsigned mask, int pred);
void note_progress();                           // an emulated state change that other fibers may be waiting for
void* dyn_smem_ptr();                           // base of the CTA's dynamic shared memory (at its window offset)
void violation(const char* fmt, ...) __attribute__((format(printf, 1, 2)));
unsigned long long virtual_ns();
void sleep_ns(unsigned ns);

struct LaunchCfg { dim3 grid, block; size_t smem; cudaStream_t stream; int cluster_x; };
void submit(const LaunchCfg& cfg, const char* name, const void* fn, std::function<void()> body);

// K<<<grid, block, smem, stream>>>(args...) is rewritten (tests/emu/build_emu.py) into
// emu::Launch(grid, block, smem, stream).run("K", K, args...)
struct Launch {
  LaunchCfg cfg;
  Launch(dim3 g, dim3 b, size_t smem = 0, cudaStream_t st = nullptr) : cfg{g, b, smem, st, 1} {}
  Launch& cluster(int x) { cfg.cluster_x = x; return *this; }
  template <class... P, class... A>
  void run(const char* name, void (*k)(P...), A&&... a) {
    std::tuple<std::decay_t<P>...> params(std::forward<A>(a)...);      // by value, as a kernel's parameters are
    submit(cfg, name, reinterpret_cast<const void*>(k), [k, params]() { std::apply(k, params); });
  }
};

}  // namespace emu

// ---- built-in variables ----
#define threadIdx (emu::cur()->tid)
#define blockIdx (emu::cur()->bid)
#define blockDim (emu::cur()->bdim)
#define gridDim (emu::cur()->gdim)

// ---- SIMT intrinsics ----
inline void __syncthreads() { emu::cta_barrier(); }
inline void __syncwarp(unsigned mask = 0xffffffffu) { emu::warp_barrier(mask); }
template <class T> inline T __shfl_sync(unsigned mask, T v, int src, int width = 32) {
  static_assert(sizeof(T) <= 8, "shuffle of at most 8 bytes");
  const int lane = emu::cur()->lane;
  const int s = (lane & ~(width - 1)) | (src & (width - 1));
  T out;
  emu::warp_exchange(mask, &v, &out, (int)sizeof(T), s);
  return out;
}
template <class T> inline T __shfl_xor_sync(unsigned mask, T v, int lanemask, int width = 32) {
  const int lane = emu::cur()->lane;
  int s = lane ^ lanemask;
  if ((s & ~(width - 1)) != (lane & ~(width - 1))) s = lane;
  T out;
  emu::warp_exchange(mask, &v, &out, (int)sizeof(T), s);
  return out;
}
template <class T> inline T __shfl_down_sync(unsigned mask, T v, unsigned delta, int width = 32) {
  const int lane = emu::cur()->lane;
  int s = lane + (int)delta;
  if ((s & ~(width - 1)) != (lane & ~(width - 1))) s = lane;
  T out;
  emu::warp_exchange(mask, &v, &out, (int)sizeof(T), s);
  return out;
}
inline unsigned __ballot_sync(unsigned mask, int pred) { return emu::warp_ballot(mask, pred); }
inline int __any_sync(unsigned mask, int pred) { return emu::warp_ballot(mask, pred) != 0; }
inline int __all_sync(unsigned mask, int pred) { return emu::warp_ballot(mask, !pred) == 0; }

inline float __uint_as_float(unsigned u) { float f; memcpy(&f, &u, 4); return f; }
inline unsigned __float_as_uint(float f) { unsigned u; memcpy(&u, &f, 4); return u; }
inline int __float_as_int(float f) { int u; memcpy(&u, &f, 4); return u; }
inline float __int_as_float(int u) { float f; memcpy(&f, &u, 4); return f; }
template <class T> inline T __ldcs(const T* p) { return *p; }
template <class T> inline T __ldg(const T* p) { return *p; }
template <class T> inline T __ldcg(const T* p) { return *p; }
inline void __threadfence() { emu::note_progress(); }
inline void __threadfence_block() {}
inline void __nanosleep(unsigned ns) { emu::sleep_ns(ns); }
inline int __popc(unsigned v) { return __builtin_popcount(v); }
inline int __ffs(int v) { return __builtin_ffs(v); }
inline int __clz(int v) { return v ? __builtin_clz((unsigned)v) : 32; }

// atomics: fibers never pre-empt one another, so plain read-modify-write is atomic here; every atomic is a state change
// another fiber may be polling for
#define EMU_ATOMIC(name, T, expr)                          \
  inline T name(T* p, T v) { const T old = *p; *p = (expr); emu::note_progress(); return old; }
EMU_ATOMIC(atomicAdd, int, old + v)
EMU_ATOMIC(atomicAdd, unsigned, old + v)
EMU_ATOMIC(atomicAdd, unsigned long long, old + v)
EMU_ATOMIC(atomicAdd, float, old + v)
EMU_ATOMIC(atomicAdd, double, old + v)
EMU_ATOMIC(atomicExch, int, v)
EMU_ATOMIC(atomicExch, unsigned, v)
EMU_ATOMIC(atomicExch, float, v)
EMU_ATOMIC(atomicOr, int, old | v)
EMU_ATOMIC(atomicOr, unsigned, old | v)
EMU_ATOMIC(atomicAnd, int, old & v)
EMU_ATOMIC(atomicMax, int, old > v ? old : v)
EMU_ATOMIC(atomicMin, int, old < v ? old : v)
#undef EMU_ATOMIC
inline int atomicCAS(int* p, int cmp, int v) { const int old = *p; if (old == cmp) *p = v; emu::note_progress(); return old; }
inline unsigned atomicCAS(unsigned* p, unsigned cmp, unsigned v) { const unsigned old = *p; if (old == cmp) *p = v; emu::note_progress(); return old; }
inline unsigned long long atomicCAS(unsigned long long* p, unsigned long long cmp, unsigned long long v) {
  const unsigned long long old = *p; if (old == cmp) *p = v; emu::note_progress(); return old;
}

using std::max;
using std::min;

// the runtime's C++ convenience overload (cuda_runtime.h provides it under nvcc only)
template <class R, class... P>
inline cudaError_t cudaFuncSetAttribute(R (*f)(P...), cudaFuncAttribute attr, int value) {
  return ::cudaFuncSetAttribute(reinterpret_cast<const void*>(f), attr, value);
}

// device-side graph API (k_loop_cond)
void cudaGraphSetConditional(cudaGraphConditionalHandle h, unsigned value);
