// kernels_tc.cu -- the tensor-core contractions of one evaluation round, sm_100a only.
//
//   k_dose_tc : d = D t (Eq. 1) on tcgen05 with a 3xTF32 split, penalty and
//               derivative (Eq. 2) and the per-plan objective partial sums
//               (Eq. 4) fused into the epilogue.  Dose never reaches HBM; the
//               epilogue emits r = dF/dd / 2 as two tf32 parts for the second contraction.
//   k_grad_tc : G = D^T r (Eq. 3 summed over points) on tcgen05, 3xTF32,
//               split over points with per-segment partial sums (fixed order, no float atomics).
//
// Tile orientation (both kernels): the 128 TMEM lanes hold 128 PLANS (MMA M = 128).
//   dose : acc[128 plans x 64 points]  = T[128 x A] (A operand) . D_chunk[64 x A]^T (B, K-major)
//          T_hi lives in TMEM for the whole kernel (A-from-TMEM MMAs), T_lo in shared memory;
//          D streams through a TMA ring in slabs of 32 dwell positions (hi and lo part).
//   grad : acc[128 plans x A]  +=  R[32 points x 128 plans]^T (A, MN-major) . D[32 points x A] (B, MN-major)
//          R and D stream through a TMA ring in slabs of 32 (or 16) points.
// 3xTF32: x = hi + lo with hi, lo representable in tf32; x.y ~ hi.hi + hi.lo + lo.hi accumulated
// in fp32 by the tensor core (the dropped lo.lo term is ~2^-22 relative).
//
// Roles (192 threads): warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer (one lane),
// warps 2-5 = epilogue (TMEM lane quadrant = warp_id % 4).  Pipelines are mbarrier rings.
#include <cudaTypedefs.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "gmco_internal.cuh"
#include "gmco_ptx.cuh"
#include "penalty.cuh"
#include "tc_layout.h"

namespace gmco {

namespace {

// Points per dose chunk = MMA N of the dose contraction (tcl::kPC).  128, not 64: a kind::tf32 M=128 K=8 MMA costs
// max(~60, N/2) cycles on sm_100 (measured, profiles/r1_mma_rate.md), so N=64 runs the tensor pipe at half rate.
using tcl::kPC; using tcl::kSlabBytes; using tcl::kTloBox; using tcl::kTmemGroups; using tcl::kScratchBytes;
using tcl::kHalfPC; using tcl::kHalfSlab; using tcl::kPairEntry;
constexpr int kThreads = 192;
static_assert(tcl::kMaxGroups * 32 == kMaxApadTensor, "tc_layout.h and gmco_internal.cuh disagree on the tensor route's limit");

// The PTX wrappers (mbarrier, TMA, tcgen05, cluster addressing) live in gmco_ptx.cuh.

// ---------------------------------------------------------------------------------------------
// Bounded waits.  A barrier that does not complete is a protocol bug; it must neither hang the GPU nor raise an SM
// exception (a trap is reported to the whole machine as Xid 13).  A wait that outlasts kWaitLimitNs writes the
// device error word (gmco_internal.cuh DevErr), raises the CTA's abort flag in shared memory and returns false; every
// other waiter of the CTA (and, through the error word, of the grid) then gives up as well, all roles fall through to
// the kernel's normal teardown (barrier, TMEM dealloc, cluster barrier) and the host reports GMCO_E_CUDA after its
// next synchronise.  The fast path is a short inline spin; the clock is only read on the slow path.
constexpr unsigned long long kWaitLimitNs = 4000000000ull;   // kernels here run for at most about a millisecond
constexpr int kFastSpins = 64;

struct Watch {
  int* err;             // device error word [4]
  uint32_t abort_addr;  // shared::cta address of this CTA's abort flag
  int kernel;           // DevErrKernel id, high byte of the reported site
};

// The slow path must not slow a healthy wait down: between two polls of the barrier it does nothing; every 64th
// failed poll it reads the CTA's abort flag (shared memory), and only every 4096th the error word (a global load) and
// the clock.  A poll takes tens of cycles at least, so the bound is checked every few tens of microseconds at most.
__device__ __noinline__ bool mbar_wait_slow(uint32_t bar, uint32_t parity, int cluster_scope, int* err, uint32_t abort_addr,
                                            int site) {
  unsigned long long t0 = 0;
  for (uint32_t spins = 1;; ++spins) {
    if (cluster_scope ? mbar_try_wait_cluster_addr(bar, parity) : mbar_try_wait_addr(bar, parity)) return true;
    if ((spins & 63u) == 0u) {
      if (ld_flag(abort_addr)) return false;
      if ((spins & 4095u) == 0u) {
        const bool failed_elsewhere = *reinterpret_cast<volatile int*>(err) != 0;
        const unsigned long long now = global_ns();
        if (t0 == 0) t0 = now;
        if (failed_elsewhere || now - t0 > kWaitLimitNs) {
          if (!failed_elsewhere && atomicCAS(err, 0, (int)DEVERR_WAIT_TIMEOUT) == 0) {
            err[1] = site; err[2] = (int)(blockIdx.x | (blockIdx.y << 16)); err[3] = (int)(threadIdx.x | (parity << 16));
          }
          st_flag(abort_addr, 1u);
          return false;
        }
      }
    }
  }
}
// The verdict is WARP-UNIFORM (a vote): every role that waits here is a whole warp in uniform control flow and goes on
// to warp-synchronous operations (elect.sync, tcgen05.ld / st .sync.aligned, __syncwarp).  Without the vote a lane that
// gave up (abort flag seen) could leave the role while a lane whose last poll still succeeded went on to wait for the
// full warp in such an operation for ever -- found by the CPU emulation of the kernels with a planted protocol error
// (tests/test_emu_mutants.py); the abort path must itself be unable to hang.
__device__ __forceinline__ bool mbar_wait_addr(const Watch& w, uint32_t bar, uint32_t parity, int site) {
  bool ok = false;
#pragma unroll 1
  for (int i = 0; i < kFastSpins && !ok; ++i) ok = mbar_try_wait_addr(bar, parity);
  if (!ok) ok = mbar_wait_slow(bar, parity, 0, w.err, w.abort_addr, (w.kernel << 8) | site);
  return __all_sync(0xffffffffu, ok) != 0;
}
__device__ __forceinline__ bool mbar_wait(const Watch& w, uint64_t* bar, uint32_t parity, int site) {
  return mbar_wait_addr(w, smem_u32(bar), parity, site);
}
// a barrier of this CTA on which threads of the peer CTA arrive (shared::cluster arrivals)
__device__ __forceinline__ bool mbar_wait_cluster(const Watch& w, uint64_t* bar, uint32_t parity, int site) {
  const uint32_t b = smem_u32(bar);
  bool ok = false;
#pragma unroll 1
  for (int i = 0; i < kFastSpins && !ok; ++i) ok = mbar_try_wait_cluster_addr(b, parity);
  if (!ok) ok = mbar_wait_slow(b, parity, 1, w.err, w.abort_addr, (w.kernel << 8) | site);
  return __all_sync(0xffffffffu, ok) != 0;       // warp-uniform, see mbar_wait_addr
}
// Waits of a role that ONE thread runs alone (the MMA issue loops: one elected lane walks the whole loop, the other
// lanes of its warp wait at the role's closing __syncwarp).  No vote, no elect and no reconvergence per ring entry:
// the fast path is one poll and one branch, everything else is out of line.  (The issuing thread's instruction stream,
// not the tensor pipe, bounds the dose kernel: profiles/r1_ncu_dose_pair.md, profiles/r2_issue_loop_sass.md.)
__device__ __forceinline__ bool mbar_wait1_addr(const Watch& w, uint32_t bar, uint32_t parity, int site) {
  if (mbar_try_wait_addr(bar, parity)) return true;
  return mbar_wait_slow(bar, parity, 0, w.err, w.abort_addr, (w.kernel << 8) | site);
}
__device__ __forceinline__ bool mbar_wait1_cluster(const Watch& w, uint64_t* bar, uint32_t parity, int site) {
  const uint32_t b = smem_u32(bar);
  if (mbar_try_wait_cluster_addr(b, parity)) return true;
  return mbar_wait_slow(b, parity, 1, w.err, w.abort_addr, (w.kernel << 8) | site);
}
// inside a role's lambda: give the role up when the wait was abandoned
#define GMCO_WAIT(call) do { if (!(call)) return; } while (0)

// Layout self-check at kernel entry: the carve-up must fit the dynamic shared memory the launch provided and the
// TMEM columns must fit 512.  A mismatch (a host/device formula drifting apart) is reported through the error word
// instead of letting a TMA write run past the CTA's window.
__device__ __forceinline__ bool layout_fits(int* err, int kernel, uint32_t pad, int smem_end, int tmem_cols) {
  const bool smem_ok = pad + (uint32_t)smem_end <= dynamic_smem_size(), tmem_ok = tmem_cols <= tcl::kTmemCols;
  if (smem_ok && tmem_ok) return true;
  if (threadIdx.x == 0 && atomicCAS(err, 0, (int)(smem_ok ? DEVERR_TMEM_LAYOUT : DEVERR_SMEM_LAYOUT)) == 0) {
    err[1] = kernel << 8; err[2] = (int)(blockIdx.x | (blockIdx.y << 16)); err[3] = smem_ok ? tmem_cols : (int)pad + smem_end;
  }
  return false;
}
// abort path of the teardown: give operations that are still in flight (TMA writes into this CTA's shared memory,
// MMAs into its TMEM) time to land before the memory is given back
__device__ __forceinline__ void drain_if_aborted(uint32_t abort_addr) {
  if (ld_flag(abort_addr)) {
    for (int i = 0; i < 200; ++i) __nanosleep(1000);
  }
}


// D[tmem] (+)= A[tmem] . B[smem]

// the two halves of smem_desc(): lo = start address | LBO, hi = SBO | version | layout
__device__ __forceinline__ uint32_t desc_lo(uint32_t saddr, uint32_t lbo_bytes) { return ((saddr >> 4) & 0x3fff) | ((lbo_bytes >> 4) << 16); }
__host__ __device__ constexpr uint32_t desc_hi(uint32_t sbo_bytes, uint32_t layout) { return (sbo_bytes >> 4) | (1u << 14) | (layout << 29); }


// Shared-memory matrix descriptor, version 1 (sm_100).  Addresses and offsets in 16 B units.
//   kSwz128 : K-major operand, rows of 128 B = 32 fp32 along K, 16 B chunks XOR-swizzled over 8 rows
//             (TMA SWIZZLE_128B).  SBO = bytes between 8-row groups (1024), LBO unused (1).
//   kSwz128Base32 : MN-major tf32 operand (the only MN-major layout tf32 has): rows of 128 B = 32 fp32
//             along M/N, one row per K index, 32 B chunks XOR-swizzled over 4 rows (TMA
//             SWIZZLE_128B_ATOM_32B).  LBO = bytes between 32-element groups along M/N,
//             SBO = bytes between 4-row groups along K (512).
constexpr uint32_t kSwz128 = 2, kSwz128Base32 = 1;
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3fff);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32;
  d |= (uint64_t)1 << 46;   // descriptor version
  d |= (uint64_t)layout << 61;
  return d;
}
// Instruction descriptor, kind::tf32, fp32 accumulator, M = 128.
__host__ __device__ constexpr uint32_t instr_desc(int n, int a_mn_major, int b_mn_major) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)a_mn_major << 15) | ((uint32_t)b_mn_major << 16) |
         ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}

struct Thresholds { float d_lo[GMCO_MAX_STRUCTS], d_hi[GMCO_MAX_STRUCTS]; };

constexpr int kDoseThreads = 320;       // warp 0 TMA, warp 1 MMA, warps 2-9 epilogue (2 per TMEM lane quadrant)

struct DoseArgs {
  const float* T;             // [K_pad][A_pad] trial dwell times, fp32; split into tf32 (hi, lo) in the prologue
  float* R;                   // [N_alloc][K_pad]  dF/dd / 2 (fp32; the gradient kernel splits it)
  float* Fpart;               // [n_tiles * segs][128][2]
  const float* Weff;          // [K_pad][2S]
  const int* tile_struct;     // [N_alloc / 64]
  const int* tile_valid;      // [N_alloc / 64]
  const int* row_src;         // [N_alloc]
  float* dose_dbg;            // [N][K] or null
  const int* gate;
  int* zero_ctr;              // start-of-round bookkeeping, done by CTA (0, 0): *zero_ctr = 0, *log_slot = *gate
  int* log_slot;
  int* round_ctr;             // counts the rounds that had a running plan (gmco_stats.rounds)
  int A_pad, K_pad, K, S, n_chunks, segs, n_stage, n_acc, sep_corr, tlo_resident;
  int tmem_groups, n_main;    // streamed layout: dwell groups of T_hi in TMEM (8, or 4 with n_main = 2 main accumulators)
  int compact_cap;            // > 0: plans are packed by slot; the CTAs re-split over the tiles that hold running plans
  int* err;                   // device error word [4] (gmco_internal.cuh DevErr); never null
  Thresholds thr;
};

struct GradArgs {
  float* Gpart;               // [n_tiles * segs][128][A_pad]
  const int* gate;
  int A_pad, n_slabs, segs, n_stage, compact_cap;
  int* err;                   // device error word [4]; never null
};

// Compaction (gmco_options.compaction): k_step packs the running plans into slots [0, n_running), so only the first
// ceil(n_running / 128) tiles hold work.  The grid is fixed (it lives in a captured graph), so its CTAs are re-dealt:
// with `ta` active tiles every tile gets min(CTAs / ta, cap) point segments.  All tiles get the same split, and the
// split depends on n_running only, so a plan's sums do not depend on which slot it was given.
__device__ __forceinline__ bool compact_remap(int n_running, int cap, int& seg, int& tile, int& segs) {
  const int ta = (n_running + 127) >> 7;
  const int total = (int)(gridDim.x * gridDim.y);
  int sa = total / ta;
  if (sa > cap) sa = cap;
  const int c = (int)(blockIdx.y * gridDim.x + blockIdx.x);
  tile = c / sa; seg = c - tile * sa; segs = sa;
  return tile < ta;
}


// ---------------------------------------------------------------------------------------------
// a2-a4 on tensor cores.  grid = (segs, n_tiles); CTA (seg, tile) owns plans [128 tile, +128) and the
// point chunks [seg n_chunks / segs, (seg + 1) n_chunks / segs).
// Shared memory: [T_lo resident: G x 16 KB]? | ring of n_stage entries | barriers.  Ring entries alternate between
// the D_hi slab and the D_lo slab of one (chunk, 32-dwell group): 16 KB each, so the ring is deep in entries although
// a chunk is 128 points wide; when T_lo is streamed, its 16 KB slab rides behind the D_hi slab of its group.
// The last kScratchBytes of the ring double as the T_hi transposition scratch of the prologue.
// kSplit (streamed layout only, gmco_options.wide_accum): two main accumulators and 4 instead of 8 dwell groups of T_hi in TMEM
template <bool kResident, bool kSplit = false>   // T_lo resident in shared memory (at most 256 dwell positions) or streamed with D_hi
__global__ void __launch_bounds__(kDoseThreads, 1)
k_dose_tc(const __grid_constant__ CUtensorMap tmD_hi, const __grid_constant__ CUtensorMap tmD_lo,
          const __grid_constant__ CUtensorMap tmT_lo, const __grid_constant__ CUtensorMap tmT, const DoseArgs a) {
  if (a.zero_ctr && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
    *a.zero_ctr = 0;
    if (a.log_slot) *a.log_slot = *a.gate;
    if (a.round_ctr && *a.gate > 0) *a.round_ctr += 1;
  }
  if (a.gate && *a.gate == 0) return;
  int seg = blockIdx.x, tile = blockIdx.y, segs = a.segs;
  if (a.compact_cap && !compact_remap(*a.gate, a.compact_cap, seg, tile, segs)) return;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int G = a.A_pad >> 5;                       // 32-dwell slabs
  // T_hi groups kept in TMEM and main accumulators: 8 / 1, or (streamed layout with gmco_options.wide_accum) 4 / 2
  static_assert(!(kResident && kSplit), "the split main accumulator belongs to the streamed layout");
  constexpr int kTg = kSplit ? tcl::kTmemGroupsSplit : kTmemGroups, n_main = kSplit ? 2 : 1;
  const tcl::DoseSmem lay = tcl::dose_smem(kResident, G, a.n_stage, kTg);
  if (!layout_fits(a.err, kResident ? DEVERR_K_DOSE_RESIDENT : DEVERR_K_DOSE_STREAMED, (uint32_t)(smem - smem_raw), lay.end,
                   tcl::dose_tmem_cols(G, kTg, n_main)))
    return;                                         // uniform over the CTA: nothing has been set up yet
  const int stageBytes = lay.stage_bytes;
  // TMEM holds T_hi of the first kTmemGroups dwell groups (256 columns); with more groups the rest of T_hi lives in
  // shared memory (the "tail", SS MMAs) so that both accumulators always fit.
  uint8_t* tlo = smem;                              // resident: T_lo [G][128 plans][128 B]; streamed: T_hi tail [G - 8][..]
  uint8_t* ring = smem + lay.ring_off;
  uint8_t* scratch = smem + lay.scratch_off;
  const int scr_slot = lay.scr_slot;                // first ring slot that overlaps the scratch
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + lay.bars_off);
  uint64_t* full = bars;                            // [n_stage]
  uint64_t* empty = bars + a.n_stage;               // [n_stage]
  uint64_t* tg_ready = bars + 2 * a.n_stage;        // [kMaxGroups]: T of dwell group g is in TMEM / smem
  uint64_t* tin_full = tg_ready + tcl::kMaxGroups;  // [kMaxGroups]: fp32 T of group g has landed (TMA)
  uint64_t* acc_full = tin_full + tcl::kMaxGroups;  // [2]
  uint64_t* acc_empty = acc_full + 2;               // [2]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + lay.slot_off);
  const Watch w{a.err, smem_u32(tmem_slot + 1), kResident ? DEVERR_K_DOSE_RESIDENT : DEVERR_K_DOSE_STREAMED};

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int c0 = (int)((long long)seg * a.n_chunks / segs), c1 = (int)((long long)(seg + 1) * a.n_chunks / segs);

  if (threadIdx.x == 0) {
    for (int i = 0; i < a.n_stage; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); }
    for (int i = 0; i < tcl::kMaxGroups; ++i) { mbar_init(tg_ready + i, 128); mbar_init(tin_full + i, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(acc_full + i, 1); mbar_init(acc_empty + i, 256); }
    tmem_slot[1] = 0u;                              // abort flag
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) { tma_prefetch_desc(&tmD_hi); tma_prefetch_desc(&tmD_lo); tma_prefetch_desc(&tmT_lo); tma_prefetch_desc(&tmT); }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = __shfl_sync(0xffffffffu, *tmem_slot, 0);   // warp-uniform for the compiler
  const uint32_t t_thi = tmem;                      // columns [0, A_pad): T_hi
  // columns [A_pad, ...): per buffer a MAIN accumulator (T_hi D_hi) and, when the columns last (A_pad <= 256), a
  // separate CORRECTION accumulator (T_hi D_lo + T_lo D_hi), 128 points each.  The tensor core truncates when it adds
  // into the fp32 accumulator; keeping the 64 small products of a chunk out of the large sum cuts that one-sided error
  // from ~1e-5 to ~2e-6 of the dose, and the dose error is what the gradient feels near a threshold (r = d - D_lim
  // cancels).  With both accumulators there is room for one buffer only: the epilogue frees it as soon as the values
  // are in registers, the penalty arithmetic and the R stores still overlap the next chunk's MMAs.
  // Split main (n_main = 2): the adds of T_hi D_hi go to accumulator A for the dwell groups below
  // g_half and to accumulator B from g_half on, so that each takes half as many truncating adds at half the
  // magnitude; the epilogue sums A + B + corrections in fp32 registers.  Columns: [main A | main B | corrections].
  const uint32_t t_acc = tmem + tcl::dose_tmem_acc_col(G, kTg);
  const int g_half = kSplit ? (G + 1) >> 1 : G;               // first dwell group of main accumulator B (none when G)
  constexpr uint32_t corr_off = (uint32_t)n_main * kPC;        // column offset of the correction accumulator

  if (warp == 0) {
    // run by ONE elected lane, like the issue loop: per ring entry one poll, expect_tx and the TMA loads
    auto producer = [&]() {
      if (c1 <= c0) return;
      const uint64_t polD = l2_evict_last(), polT = l2_evict_normal();
      if (kResident) {                         // fp32 T of the tile lands where its lo part will live
        {
          for (int g = 0; g < G; ++g) {
            mbar_expect_tx(tin_full + g, (uint32_t)kTloBox);
            tma_load_3d(&tmT, tlo + (size_t)g * kTloBox, tin_full + g, 0, tile * 128, g, polT);
          }
        }
      }
      int st = 0; uint32_t ph = 0;
      bool scratch_busy = !kResident;          // resident mode transposes through the T_lo area itself
      for (int c = c0; c < c1; ++c) {
        for (int g2 = 0; g2 < 2 * G; ++g2) {          // entry 2 g: D_hi (+ streamed T_lo), entry 2 g + 1: D_lo
          const int g = g2 >> 1, lo = g2 & 1;
          if (scratch_busy && st >= scr_slot) {       // the prologue's transposition scratch overlaps these slots
            for (int i = 0; i < G; ++i) GMCO_WAIT(mbar_wait1_addr(w, smem_u32(tg_ready + i), 0, DEVERR_W_TG_READY));
            scratch_busy = false;
          }
          GMCO_WAIT(mbar_wait1_addr(w, smem_u32(empty + st), ph ^ 1, DEVERR_W_EMPTY));
          {
            uint8_t* dst = ring + (size_t)st * stageBytes;
            const bool with_t = !lo && !kResident;
            mbar_expect_tx(full + st, (uint32_t)(with_t ? kSlabBytes + kTloBox : kSlabBytes));
            tma_load_3d(lo ? &tmD_lo : &tmD_hi, dst, full + st, 0, c * kPC, g, polD);
            if (with_t) tma_load_3d(&tmT_lo, dst + kSlabBytes, full + st, 0, tile * 128, g, polT);
          }
          if (++st == a.n_stage) { st = 0; ph ^= 1; }
        }
      }
    };
    if (elect_one()) producer();                      // one lane issues every TMA load of the CTA
    __syncwarp();
  } else if (warp == 1) {
    auto issuer = [&]() {
      if (c1 <= c0) return;
      // Issue loop, run by ONE elected lane (see below): per ring entry one poll of the full barrier, 8 or 4 MMAs whose
      // descriptors differ by 32-bit adds, one commit -- no vote, elect or reconvergence per entry.
      constexpr uint32_t idesc = instr_desc(kPC, 0, 0);
      constexpr uint32_t dhi = desc_hi(1024, kSwz128);
      const int n_stage = a.n_stage, n_acc = a.n_acc;
      const uint32_t ring_lo = desc_lo(smem_u32(ring), 16), ring_step = (uint32_t)stageBytes >> 4;
      const uint32_t tlo_lo0 = desc_lo(smem_u32(tlo), 16);
      const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty);
      int st = 0; uint32_t ph = 0;
      for (int c = c0; c < c1; ++c) {
        const int b = n_acc == 2 ? (c - c0) & 1 : 0, use = n_acc == 2 ? (c - c0) >> 1 : c - c0;
        GMCO_WAIT(mbar_wait1_addr(w, smem_u32(acc_empty + b), (use & 1) ^ 1, DEVERR_W_ACC_EMPTY));
        tc_fence_after();
        const uint32_t acc0 = t_acc + b * (a.sep_corr ? (uint32_t)(n_main + 1) * kPC : kPC), acc_c = a.sep_corr ? acc0 + corr_off : acc0;
        uint32_t thi = t_thi, alo = tlo_lo0;   // alo: resident T_lo slab g, or (streamed) T_hi tail slab g - kTg
        for (int g = 0; g < G; thi += 32, alo += (kResident || g >= kTg) ? kTloBox >> 4 : 0, ++g) {
          // entry 2 g: D_hi slab (+ the streamed T_lo slab behind it): T_hi D_hi and T_lo D_hi
          if (c == c0) { GMCO_WAIT(mbar_wait1_addr(w, smem_u32(tg_ready + g), 0, DEVERR_W_TG_READY)); tc_fence_after(); }   // first chunk overlaps the prologue
          GMCO_WAIT(mbar_wait1_addr(w, full0 + 8 * st, ph, DEVERR_W_FULL));
          {
            const uint32_t bd = ring_lo + (uint32_t)st * ring_step;
            const uint32_t ad = kResident ? alo : bd + (kSlabBytes >> 4);
            const uint32_t acc = g < g_half ? acc0 : acc0 + kPC;                 // main accumulator A or B
            const uint32_t first = (g != 0 && g != g_half) ? 1u : 0u;           // the first add into A / into B overwrites
            if (kResident || g < kTg) {
              mma_ts2(acc, thi, bd, dhi, idesc, first);
              mma_ss2(acc_c, ad, dhi, bd, dhi, idesc, (a.sep_corr && g == 0) ? 0u : 1u);
#pragma unroll
              for (int j = 1; j < 4; ++j) {         // K-steps of 8 dwell positions: +32 B inside the swizzled row
                mma_ts2(acc, thi + 8 * j, bd + 2 * j, dhi, idesc, 1);
                mma_ss2(acc_c, ad + 2 * j, dhi, bd + 2 * j, dhi, idesc, 1);
              }
            } else {                                // T_hi of this group is in the shared-memory tail
              mma_ss2(acc, alo, dhi, bd, dhi, idesc, first);
              mma_ss2(acc_c, ad, dhi, bd, dhi, idesc, 1);
#pragma unroll
              for (int j = 1; j < 4; ++j) {
                mma_ss2(acc, alo + 2 * j, dhi, bd + 2 * j, dhi, idesc, 1);
                mma_ss2(acc_c, ad + 2 * j, dhi, bd + 2 * j, dhi, idesc, 1);
              }
            }
            tc_commit_addr(empty0 + 8 * st);
          }
          if (++st == n_stage) { st = 0; ph ^= 1; }
          // entry 2 g + 1: D_lo slab: T_hi D_lo
          GMCO_WAIT(mbar_wait1_addr(w, full0 + 8 * st, ph, DEVERR_W_FULL));
          {
            const uint32_t bd = ring_lo + (uint32_t)st * ring_step;
            if (kResident || g < kTg) {
#pragma unroll
              for (int j = 0; j < 4; ++j) mma_ts2(acc_c, thi + 8 * j, bd + 2 * j, dhi, idesc, 1);
            } else {
#pragma unroll
              for (int j = 0; j < 4; ++j) mma_ss2(acc_c, alo + 2 * j, dhi, bd + 2 * j, dhi, idesc, 1);
            }
            tc_commit_addr(empty0 + 8 * st);
            if (g == G - 1) tc_commit(acc_full + b);
          }
          if (++st == n_stage) { st = 0; ph ^= 1; }
        }
      }
    };
    if (elect_one()) issuer();                        // one lane issues every MMA and commit of the CTA
    __syncwarp();
  } else {
    const int e = warp - 2;                         // 0..7
    const int q = warp & 3;                         // TMEM lane quadrant this warp may access
    const int h = e >> 2;                           // which 32 of the chunk's 64 points this warp evaluates
    const int L = q * 32 + lane;                    // lane = plan inside the tile
    const int plan = tile * 128 + L;
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    float f_lo = 0.f, f_hi = 0.f;
    auto epilogue = [&]() {
      if (c1 <= c0) return;
      // Prologue: the tile's trial dwell times T (fp32, read ONCE) are split here into tf32 parts: hi -> TMEM columns
      // [0, A_pad) (the A operand of T_hi D), lo -> shared memory (the A operand of T_lo D_hi).  Slabs g = h, h + 2, ...;
      // each slab has its own ready barrier, so the first chunk's MMAs start while later slabs are still on their way.
      if (kResident) {
        // TMA has put slab g of T where T_lo will live, in the SWIZZLE_128B K-major layout of the MMA descriptor.
        // Thread = plan row: it reads its own 128 B row (8 swizzled 16 B chunks), keeps hi for TMEM and writes lo
        // back in place -- no cross-thread hand-off, no transposition scratch.
        const int row = q * 32 + lane;
        for (int g = h; g < G; g += 2) {
          uint8_t* base = tlo + (size_t)g * kTloBox + row * 128;
          GMCO_WAIT(mbar_wait(w, tin_full + g, 0, DEVERR_W_TIN_FULL));
          uint32_t v[32];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            float4* cell = reinterpret_cast<float4*>(base + ((k ^ (row & 7)) << 4));
            const float4 t = *cell;
            float4 hi, lo;
            hi.x = tf32_rn(t.x); hi.y = tf32_rn(t.y); hi.z = tf32_rn(t.z); hi.w = tf32_rn(t.w);
            lo.x = tf32_rn(t.x - hi.x); lo.y = tf32_rn(t.y - hi.y); lo.z = tf32_rn(t.z - hi.z); lo.w = tf32_rn(t.w - hi.w);
            *cell = lo;
            v[4 * k + 0] = __float_as_uint(hi.x); v[4 * k + 1] = __float_as_uint(hi.y);
            v[4 * k + 2] = __float_as_uint(hi.z); v[4 * k + 3] = __float_as_uint(hi.w);
          }
          tmem_st32(t_thi + lane_base + g * 32, v);
          tmem_st_wait();
          tc_fence_before();
          fence_proxy_async();                      // the lo stores above are read by the MMA (async proxy)
          mbar_arrive(tg_ready + g);
        }
      } else {
        // streamed-T_lo mode (more than 256 dwell positions): T_lo comes from global memory with every D_hi slab;
        // hi is read from T with coalesced 128 B row loads and transposed through the tail of the ring.
        uint8_t* scr = scratch + e * 4096;
        const int r0 = lane >> 3, c4 = lane & 7;
        const float* src = a.T + (size_t)(tile * 128 + q * 32) * a.A_pad;
        for (int g = h; g < G; g += 2) {
          float4 t[8];
#pragma unroll
          for (int i = 0; i < 8; ++i)
            t[i] = *reinterpret_cast<const float4*>(src + (size_t)(i * 4 + r0) * a.A_pad + g * 32 + c4 * 4);
          if (g >= kTg) {                            // tail group: hi goes to shared memory in the operand layout
            uint8_t* dstg = tlo + (size_t)(g - kTg) * kTloBox + q * 4096;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int r = i * 4 + r0;
              float4 hi;
              hi.x = tf32_rn(t[i].x); hi.y = tf32_rn(t[i].y); hi.z = tf32_rn(t[i].z); hi.w = tf32_rn(t[i].w);
              *reinterpret_cast<float4*>(dstg + r * 128 + ((c4 ^ (r & 7)) << 4)) = hi;
            }
            fence_proxy_async();
            mbar_arrive(tg_ready + g);
            continue;
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int r = i * 4 + r0;
            float4 hi;
            hi.x = tf32_rn(t[i].x); hi.y = tf32_rn(t[i].y); hi.z = tf32_rn(t[i].z); hi.w = tf32_rn(t[i].w);
            *reinterpret_cast<float4*>(scr + r * 128 + ((c4 ^ (r & 7)) << 4)) = hi;
          }
          __syncwarp();
          uint32_t v[32];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const float4 u = *reinterpret_cast<const float4*>(scr + lane * 128 + ((k ^ (lane & 7)) << 4));
            v[4 * k + 0] = __float_as_uint(u.x); v[4 * k + 1] = __float_as_uint(u.y);
            v[4 * k + 2] = __float_as_uint(u.z); v[4 * k + 3] = __float_as_uint(u.w);
          }
          __syncwarp();
          tmem_st32(t_thi + lane_base + g * 32, v);
          tmem_st_wait();
          tc_fence_before();
          mbar_arrive(tg_ready + g);
        }
      }

      // This warp evaluates the 64-row tile 2 c + h of chunk c (one structure per 64-row tile by construction).
      // Structure id, valid rows and weights of the NEXT chunk are fetched one chunk ahead.
      int s_n = a.tile_struct[2 * c0 + h], nv_n = a.tile_valid[2 * c0 + h];
      float wlo_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n], whi_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n + 1];
      for (int c = c0; c < c1; ++c) {
        const int b = a.n_acc == 2 ? (c - c0) & 1 : 0, use = a.n_acc == 2 ? (c - c0) >> 1 : c - c0;
        const int s = s_n, nv = nv_n;
        const float wlo = wlo_n, whi = whi_n;
        if (c + 1 < c1) {
          s_n = a.tile_struct[2 * (c + 1) + h]; nv_n = a.tile_valid[2 * (c + 1) + h];
          wlo_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n]; whi_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n + 1];
        }
        const float dlo = a.thr.d_lo[s], dhi = a.thr.d_hi[s];
        GMCO_WAIT(mbar_wait(w, acc_full + b, use & 1, DEVERR_W_ACC_FULL));
        tc_fence_after();
        uint32_t v[2][32];
        const uint32_t t_main = t_acc + lane_base + b * (a.sep_corr ? (uint32_t)(n_main + 1) * kPC : kPC) + h * 64;
        tmem_ld32(t_main, v[0]);
        tmem_ld32(t_main + 32, v[1]);
        if (a.sep_corr) {
#pragma unroll
          for (int part = 1; part <= n_main; ++part) {       // main accumulator B (split main), then the corrections
#pragma unroll
            for (int sub = 0; sub < 2; ++sub) {
              uint32_t vc[32];
              tmem_ld32(t_main + (uint32_t)part * kPC + sub * 32, vc);
              tmem_ld_wait();
#pragma unroll
              for (int j = 0; j < 32; ++j) v[sub][j] = __float_as_uint(__uint_as_float(v[sub][j]) + __uint_as_float(vc[j]));
            }
          }
        } else {
          tmem_ld_wait();
        }
        // hand the accumulator back: tcgen05.wait::ld above, fence, then a RELEASING arrive (the documented pattern;
        // .release.cta costs no memory barrier beyond the CTA)
        tc_fence_before();
        mbar_arrive(acc_empty + b);
#pragma unroll
        for (int sub = 0; sub < 2; ++sub) {
          const int nvh = nv - sub * 32;
          const size_t p0 = (size_t)c * kPC + h * 64 + sub * 32;
          float* rp = a.R + p0 * a.K_pad + plan;
          if (nvh >= 32) {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const float d = __uint_as_float(v[sub][j]);
              rp[(size_t)j * a.K_pad] = eq2_accumulate<float>(d, dlo, dhi, wlo, whi, f_lo, f_hi);  // = dF/dd / 2
            }
          } else {                                                          // ragged tail of a structure
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const float d = __uint_as_float(v[sub][j]);
              float t_lo = f_lo, t_hi = f_hi;
              rp[(size_t)j * a.K_pad] = eq2_accumulate<float>(d, dlo, dhi, wlo, whi, t_lo, t_hi);  // padding rows: value unused
              if (j < nvh) { f_lo = t_lo; f_hi = t_hi; }
            }
          }
          if (a.dose_dbg && plan < a.K) {
            for (int j = 0; j < 32; ++j) {
              if (j < nvh) a.dose_dbg[(size_t)a.row_src[p0 + j] * a.K + plan] = __uint_as_float(v[sub][j]);
            }
          }
        }
      }
    };
    epilogue();
    a.Fpart[(((size_t)tile * segs + seg) * 128 + L) * 2 + h] = f_lo + f_hi;
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { drain_if_aborted(w.abort_addr); tc_fence_after(); tmem_dealloc(tmem, 512); }
}

// ---------------------------------------------------------------------------------------------
// a2-a4 on tensor cores, CTA-PAIR variant (tcgen05 cta_group::2).  The two CTAs of a cluster (2, 1, 1) own two adjacent
// plan tiles and the SAME point chunks.  One MMA spans both: M = 256 plans (128 TMEM lanes in each CTA, each CTA's own
// T_hi in its TMEM and T_lo in its shared memory), N = 128 points whose D slab is split between the two CTAs'
// shared memories (64 points = 8 KB each).  Every CTA therefore loads HALF of each D slab: the operand stream from L2,
// which is what kept k_dose_tc off the MMA floor, halves, and the same ring bytes hold twice as many
// entries.  Only the leader (cluster rank 0) issues MMAs; its `full` barriers collect the bytes of both CTAs' TMA
// loads, its tg_ready / acc_empty barriers the arrivals of both CTAs' epilogue threads; MMA completion is committed
// to both CTAs' `empty` / `acc_full` barriers by multicast.  Resident-T_lo layout only (at most 256 dwell positions).
// kind::tf32, fp32 accumulator, M = 256 across the pair
__host__ __device__ constexpr uint32_t instr_desc_pair(int n) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}
// compaction with pairs: the grid's CTA PAIRS are re-dealt over the active tile pairs (cf. compact_remap)
__device__ __forceinline__ bool compact_remap_pair(int n_running, int cap, int rank, int& seg, int& tile, int& segs) {
  const int tap = (((n_running + 127) >> 7) + 1) >> 1;
  const int total = (int)(gridDim.y * (gridDim.x >> 1));
  int sa = total / tap;
  if (sa > cap) sa = cap;
  const int c = (int)(blockIdx.y * (gridDim.x >> 1) + (blockIdx.x >> 1));
  const int pt = c / sa;
  tile = 2 * pt + rank; seg = c - pt * sa; segs = sa;
  return pt < tap;
}

template <int GP, int NS>   // GP > 0: ceil(A_pad / 64) and the ring size are compile-time (static issue schedule); 0: any shape
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kDoseThreads, 1)
k_dose_tc_pair(const __grid_constant__ CUtensorMap tmD_hi, const __grid_constant__ CUtensorMap tmD_lo,
               const __grid_constant__ CUtensorMap tmT, const DoseArgs a) {
  if (a.zero_ctr && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
    *a.zero_ctr = 0;
    if (a.log_slot) *a.log_slot = *a.gate;
    if (a.round_ctr && *a.gate > 0) *a.round_ctr += 1;
  }
  if (a.gate && *a.gate == 0) return;                 // both CTAs of a pair take every early exit together
  const int rank = (int)cluster_ctarank();
  const bool leader = rank == 0;
  int seg = blockIdx.y, tile = blockIdx.x, segs = a.segs;   // grid (tiles, segs): a 2-CTA MMA pair must be adjacent in x
  if (a.compact_cap && !compact_remap_pair(*a.gate, a.compact_cap, rank, seg, tile, segs)) return;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int G = a.A_pad >> 5;                         // 32-dwell groups, at most kTmemGroups
  const tcl::PairSmem lay = tcl::pair_smem(G, a.n_stage);
  // the same numbers in both CTAs of the pair (same launch, same shape): they leave together or not at all
  if (!layout_fits(a.err, DEVERR_K_DOSE_PAIR, (uint32_t)(smem - smem_raw), lay.end, tcl::pair_tmem_cols(G))) return;
  uint8_t* tlo = smem;                                // T_lo [G][128 plans][128 B]
  uint8_t* ring = smem + lay.ring_off;                // n_stage entries of two half slabs
  const int Gp = (G + 1) >> 1;                        // entries per pass over the dwell groups (a missing odd group is zero-filled)
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + lay.bars_off);
  uint64_t* full = bars;                              // [n_stage]  used in the leader: both CTAs' bytes
  uint64_t* empty = bars + a.n_stage;                 // [n_stage]  in each CTA: multicast commit
  uint64_t* tg_ready = bars + 2 * a.n_stage;          // [8]        used in the leader: 256 arrivals (both CTAs)
  uint64_t* tin_full = tg_ready + kTmemGroups;        // [8]        in each CTA: its own T
  uint64_t* acc_full = tin_full + kTmemGroups;        // [2]        in each CTA: multicast commit
  uint64_t* acc_empty = acc_full + 2;                 // [2]        used in the leader: 512 arrivals
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + lay.slot_off);
  const Watch w{a.err, smem_u32(tmem_slot + 1), DEVERR_K_DOSE_PAIR};

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int c0 = (int)((long long)seg * a.n_chunks / segs), c1 = (int)((long long)(seg + 1) * a.n_chunks / segs);

  if (threadIdx.x == 0) {
    for (int i = 0; i < a.n_stage; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); }
    for (int i = 0; i < kTmemGroups; ++i) { mbar_init(tg_ready + i, 256); mbar_init(tin_full + i, 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(acc_full + i, 1); mbar_init(acc_empty + i, 512); }
    tmem_slot[1] = 0u;                                // abort flag
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) { tma_prefetch_desc(&tmD_hi); tma_prefetch_desc(&tmD_lo); tma_prefetch_desc(&tmT); }
  if (warp == 1) tmem_alloc_pair(tmem_slot, 512);
  tc_fence_before();
  cluster_sync_all();                                 // barriers of both CTAs exist before anything arrives on them
  tc_fence_after();
  const uint32_t tmem = __shfl_sync(0xffffffffu, *tmem_slot, 0);
  const uint32_t t_thi = tmem;                        // columns [0, A_pad): T_hi
  // Two accumulator buffers of 128 points.  ONE accumulator per chunk takes all three products, the small ones first:
  // the tensor core truncates when it adds into the fp32 accumulator, so T_hi D_lo + T_lo D_hi (2^-11 of the dose) are
  // summed while the accumulator is still small and the 4 G adds of T_hi D_hi come last -- the same one-sided error as
  // with k_dose_tc's separate correction accumulator, in half the columns, which is what lets the epilogue of chunk c
  // overlap the MMAs of chunk c + 1.  The price is a second pass over the chunk's D_hi slabs (3 G ring entries per
  // chunk instead of 2 G), affordable here because every CTA loads half slabs.
  const uint32_t t_acc = tmem + G * 32;

  if (warp == 0) {
    auto producer = [&]() {
      if (c1 <= c0) return;
      const uint64_t polD = l2_evict_last(), polT = l2_evict_normal();
      {
        for (int g = 0; g < G; ++g) {
          mbar_expect_tx(tin_full + g, (uint32_t)kTloBox);
          tma_load_3d(&tmT, tlo + (size_t)g * kTloBox, tin_full + g, 0, tile * 128, g, polT);
        }
      }
      const uint32_t lfull0 = leader_addr(full), empty0 = smem_u32(empty);
      const int n_stage = a.n_stage;
      int st = 0; uint32_t ph = 0;
      // one ring entry: this CTA's half (64 points) of two dwell groups of a D slab; the bytes count on the LEADER's barrier
      auto load = [&](const CUtensorMap* map, const int c, const int gp) -> bool {
        if (!mbar_wait1_addr(w, empty0 + 8u * (uint32_t)st, ph ^ 1, DEVERR_W_EMPTY)) return false;
        if (leader) mbar_expect_tx(full + st, 2u * (uint32_t)kPairEntry);
        tma_load_3d_pair(map, ring + (size_t)st * kPairEntry, lfull0 + 8u * (uint32_t)st, 0, c * kPC + rank * kHalfPC, 2 * gp, polD);
        if (++st == n_stage) { st = 0; ph ^= 1; }
        return true;
      };
      for (int c = c0; c < c1; ++c) {
        for (int gp = 0; gp < Gp; ++gp) {             // entries 2 p, 2 p + 1: D_lo, D_hi (corrections)
          GMCO_WAIT(load(&tmD_lo, c, gp));
          GMCO_WAIT(load(&tmD_hi, c, gp));
        }
        for (int gp = 0; gp < Gp; ++gp) GMCO_WAIT(load(&tmD_hi, c, gp));   // entries 2 Gp + p: D_hi again (main product)
      }
    };
    if (elect_one()) producer();                      // one lane issues every TMA load of the CTA
    __syncwarp();
  } else if (warp == 1) {
    auto issuer = [&]() {
      if (!leader || c1 <= c0) return;
      constexpr uint32_t idesc = instr_desc_pair(kPC);
      constexpr uint32_t dhi = desc_hi(1024, kSwz128);
      const int n_stage = a.n_stage;
      const uint32_t ring_lo = desc_lo(smem_u32(ring), 16), ring_step = (uint32_t)kPairEntry >> 4;
      const uint32_t tlo_lo0 = desc_lo(smem_u32(tlo), 16);
      const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty);
      constexpr uint32_t kG1 = (uint32_t)kHalfSlab >> 4;       // second dwell group of an entry
      // This whole role is run by ONE elected lane (see below).  One ring entry: wait, 4 or 8 MMAs, commit.  kind 0: T_hi D_lo, 1: T_lo D_hi, 2: T_hi D_hi.  false: wait abandoned.
      auto entry = [&](const int kind, const int gp, const int st, const uint32_t ph, const uint32_t acc, const bool two,
                       const uint32_t acc_full_bar) -> bool {
        if (!mbar_wait1_addr(w, full0 + 8 * st, ph, DEVERR_W_FULL)) return false;
        tc_fence_after();
        {
          const uint32_t bd = ring_lo + (uint32_t)st * ring_step;
          const uint32_t thi = t_thi + 64 * gp, alo = tlo_lo0 + 2 * (kTloBox >> 4) * gp;
          if (kind == 1) {
#pragma unroll
            for (int j = 0; j < 4; ++j) mma_ss2_pair(acc, alo + 2 * j, dhi, bd + 2 * j, dhi, idesc, 1);
            if (two) {
#pragma unroll
              for (int j = 0; j < 4; ++j) mma_ss2_pair(acc, alo + (kTloBox >> 4) + 2 * j, dhi, bd + kG1 + 2 * j, dhi, idesc, 1);
            }
          } else {
            mma_ts2_pair(acc, thi, bd, dhi, idesc, (kind == 0 && gp == 0) ? 0u : 1u);
#pragma unroll
            for (int j = 1; j < 4; ++j) mma_ts2_pair(acc, thi + 8 * j, bd + 2 * j, dhi, idesc, 1);
            if (two) {
#pragma unroll
              for (int j = 0; j < 4; ++j) mma_ts2_pair(acc, thi + 32 + 8 * j, bd + kG1 + 2 * j, dhi, idesc, 1);
            }
          }
          tc_commit_pair(empty0 + 8 * st);
          if (acc_full_bar) tc_commit_pair(acc_full_bar);
        }
        return true;
      };
      if constexpr (GP > 0) {
        // Static schedule: 3 GP entries per chunk go round a ring of NS entries a whole number of times, so every
        // entry's ring slot is a compile-time constant and its phase is one bit toggled per chunk.
        constexpr int E = 3 * GP, REV = E / NS;
        static_assert(E % NS == 0, "ring size must divide the entries of a chunk");
        uint32_t chunk_par = 0;
        const bool odd = (G & 1) != 0;
        for (int c = c0; c < c1; ++c) {
          const int b = (c - c0) & 1, use = (c - c0) >> 1;
          GMCO_WAIT(mbar_wait1_cluster(w, acc_empty + b, (use & 1) ^ 1, DEVERR_W_ACC_EMPTY));
          tc_fence_after();
          const uint32_t acc = t_acc + (uint32_t)b * kPC;
#pragma unroll
          for (int gp = 0; gp < GP; ++gp) {
            const bool two = gp < GP - 1 || !odd;
            if (c == c0) {                            // the first chunk overlaps the prologue, group by group
              GMCO_WAIT(mbar_wait1_cluster(w, tg_ready + 2 * gp, 0, DEVERR_W_TG_READY));
              if (two) GMCO_WAIT(mbar_wait1_cluster(w, tg_ready + 2 * gp + 1, 0, DEVERR_W_TG_READY));
              tc_fence_after();
            }
            GMCO_WAIT(entry(0, gp, (2 * gp) % NS, chunk_par ^ (((2 * gp) / NS) & 1), acc, two, 0u));
            GMCO_WAIT(entry(1, gp, (2 * gp + 1) % NS, chunk_par ^ (((2 * gp + 1) / NS) & 1), acc, two, 0u));
          }
#pragma unroll
          for (int gp = 0; gp < GP; ++gp) {
            const bool two = gp < GP - 1 || !odd;
            GMCO_WAIT(entry(2, gp, (2 * GP + gp) % NS, chunk_par ^ (((2 * GP + gp) / NS) & 1), acc, two,
                            gp == GP - 1 ? smem_u32(acc_full + b) : 0u));
          }
          chunk_par ^= (uint32_t)(REV & 1);
        }
      } else {
        int st = 0; uint32_t ph = 0;
        for (int c = c0; c < c1; ++c) {
          const int b = (c - c0) & 1, use = (c - c0) >> 1;
          GMCO_WAIT(mbar_wait1_cluster(w, acc_empty + b, (use & 1) ^ 1, DEVERR_W_ACC_EMPTY));
          tc_fence_after();
          const uint32_t acc = t_acc + (uint32_t)b * kPC;
          for (int gp = 0; gp < Gp; ++gp) {           // corrections first
            const bool two = 2 * gp + 1 < G;
            if (c == c0) {
              GMCO_WAIT(mbar_wait1_cluster(w, tg_ready + 2 * gp, 0, DEVERR_W_TG_READY));
              if (two) GMCO_WAIT(mbar_wait1_cluster(w, tg_ready + 2 * gp + 1, 0, DEVERR_W_TG_READY));
              tc_fence_after();
            }
            GMCO_WAIT(entry(0, gp, st, ph, acc, two, 0u));
            if (++st == n_stage) { st = 0; ph ^= 1; }
            GMCO_WAIT(entry(1, gp, st, ph, acc, two, 0u));
            if (++st == n_stage) { st = 0; ph ^= 1; }
          }
          for (int gp = 0; gp < Gp; ++gp) {           // then the large product: D_hi again
            GMCO_WAIT(entry(2, gp, st, ph, acc, 2 * gp + 1 < G, gp == Gp - 1 ? smem_u32(acc_full + b) : 0u));
            if (++st == n_stage) { st = 0; ph ^= 1; }
          }
        }
      }
    };
    if (elect_one()) issuer();                        // one lane issues every MMA and commit of the CTA pair
    __syncwarp();
  } else {
    const int e = warp - 2;                           // 0..7
    const int q = warp & 3;                           // TMEM lane quadrant this warp may access
    const int h = e >> 2;                             // which 64 of the chunk's 128 points this warp evaluates
    const int L = q * 32 + lane;                      // lane = plan inside the tile
    const int plan = tile * 128 + L;
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    float f_lo = 0.f, f_hi = 0.f;
    auto epilogue = [&]() {
      if (c1 <= c0) return;
      const uint32_t l_tg = leader_addr(tg_ready), l_ae = leader_addr(acc_empty);
      // prologue: split this CTA's T into tf32 hi (TMEM) and lo (in place), as in k_dose_tc<true>
      const int row = q * 32 + lane;
      for (int g = h; g < G; g += 2) {
        uint8_t* base = tlo + (size_t)g * kTloBox + row * 128;
        GMCO_WAIT(mbar_wait(w, tin_full + g, 0, DEVERR_W_TIN_FULL));
        uint32_t v[32];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          float4* cell = reinterpret_cast<float4*>(base + ((k ^ (row & 7)) << 4));
          const float4 t = *cell;
          float4 hi, lo;
          hi.x = tf32_rn(t.x); hi.y = tf32_rn(t.y); hi.z = tf32_rn(t.z); hi.w = tf32_rn(t.w);
          lo.x = tf32_rn(t.x - hi.x); lo.y = tf32_rn(t.y - hi.y); lo.z = tf32_rn(t.z - hi.z); lo.w = tf32_rn(t.w - hi.w);
          *cell = lo;
          v[4 * k + 0] = __float_as_uint(hi.x); v[4 * k + 1] = __float_as_uint(hi.y);
          v[4 * k + 2] = __float_as_uint(hi.z); v[4 * k + 3] = __float_as_uint(hi.w);
        }
        tmem_st32(t_thi + lane_base + g * 32, v);
        tmem_st_wait();
        tc_fence_before();
        fence_proxy_async();                          // the lo stores above are read by the MMA (async proxy)
        mbar_arrive_cluster(l_tg + 8u * (uint32_t)g);
      }

      int s_n = a.tile_struct[2 * c0 + h], nv_n = a.tile_valid[2 * c0 + h];
      float wlo_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n], whi_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n + 1];
      for (int c = c0; c < c1; ++c) {
        const int s = s_n, nv = nv_n;
        const float wlo = wlo_n, whi = whi_n;
        if (c + 1 < c1) {
          s_n = a.tile_struct[2 * (c + 1) + h]; nv_n = a.tile_valid[2 * (c + 1) + h];
          wlo_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n]; whi_n = a.Weff[(size_t)plan * 2 * a.S + 2 * s_n + 1];
        }
        const float dlo = a.thr.d_lo[s], dhi = a.thr.d_hi[s];
        const int b = (c - c0) & 1, use = (c - c0) >> 1;
        GMCO_WAIT(mbar_wait(w, acc_full + b, use & 1, DEVERR_W_ACC_FULL));
        tc_fence_after();
        uint32_t v[2][32];
        const uint32_t t_main = t_acc + lane_base + (uint32_t)b * kPC + h * 64;
        tmem_ld32(t_main, v[0]);
        tmem_ld32(t_main + 32, v[1]);
        tmem_ld_wait();
        // hand the accumulator back to the leader: tcgen05.wait::ld above, fence, then a RELEASING arrive at cluster
        // scope (the documented pattern; the R stores of this chunk come after it and are not held up by it)
        tc_fence_before();
        mbar_arrive_cluster(l_ae + 8u * (uint32_t)b);
#pragma unroll
        for (int sub = 0; sub < 2; ++sub) {
          const int nvh = nv - sub * 32;
          const size_t p0 = (size_t)c * kPC + h * 64 + sub * 32;
          float* rp = a.R + p0 * a.K_pad + plan;
          if (nvh >= 32) {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const float d = __uint_as_float(v[sub][j]);
              rp[(size_t)j * a.K_pad] = eq2_accumulate<float>(d, dlo, dhi, wlo, whi, f_lo, f_hi);  // = dF/dd / 2
            }
          } else {                                                          // ragged tail of a structure
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const float d = __uint_as_float(v[sub][j]);
              float t_lo = f_lo, t_hi = f_hi;
              rp[(size_t)j * a.K_pad] = eq2_accumulate<float>(d, dlo, dhi, wlo, whi, t_lo, t_hi);  // padding rows: value unused
              if (j < nvh) { f_lo = t_lo; f_hi = t_hi; }
            }
          }
          if (a.dose_dbg && plan < a.K) {
            for (int j = 0; j < 32; ++j) {
              if (j < nvh) a.dose_dbg[(size_t)a.row_src[p0 + j] * a.K + plan] = __uint_as_float(v[sub][j]);
            }
          }
        }
      }
    };
    epilogue();
    a.Fpart[(((size_t)tile * segs + seg) * 128 + L) * 2 + h] = f_lo + f_hi;
  }
  tc_fence_before();
  if (warp == 1) drain_if_aborted(w.abort_addr);      // before the peer may tear down as well
  cluster_sync_all();                                 // neither CTA's shared memory, TMEM or barriers may go before both are done
  if (warp == 1) { tc_fence_after(); tmem_dealloc_pair(tmem, 512); }
}

// ---------------------------------------------------------------------------------------------
// a5 on tensor cores.  grid = (segs, n_tiles); CTA (seg, tile) owns plans [128 tile, +128) and the
// point slabs [seg n_slabs / segs, (seg + 1) n_slabs / segs) of PS points each.
// Stage = [R | R_lo | D_hi | D_lo]: TMA brings R (fp32), D_hi, D_lo; warps 2-5 split R in place into its
// tf32 parts (hi = truncation, lo = r - hi) before the MMA warp may read the stage.
// D_hi / D_lo come pre-split from memory (csrc/gmco_api.cu splits D once per case): deriving D_lo in these warps would
// save 16 KB of TMA per stage but add 32 KB of shared-memory reads + writes to a stage that already moves 136 KB
// through shared memory in 768 tensor-pipe cycles.
template <int PS>
__global__ void __launch_bounds__(kThreads, 1)
k_grad_tc(const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmD_hi,
          const __grid_constant__ CUtensorMap tmD_lo, const GradArgs a) {
  if (a.gate && *a.gate == 0) return;
  int seg = blockIdx.x, tile = blockIdx.y, segs = a.segs;
  if (a.compact_cap && !compact_remap(*a.gate, a.compact_cap, seg, tile, segs)) return;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem0 = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int G = a.A_pad >> 5;
  const tcl::GradSmem lay = tcl::grad_smem(PS, G, a.n_stage);
  if (!layout_fits(a.err, DEVERR_K_GRAD, (uint32_t)(smem0 - smem_raw), lay.end, tcl::grad_tmem_cols(a.A_pad))) return;
  uint8_t* smem = smem0 + lay.ring_off;             // [barriers 1 KB | ring | (epilogue row staging may run past the ring)]
  constexpr int kRBytes = 4 * PS * 128;             // R part: 4 plan groups x PS points x 128 B
  const int dBytes = lay.d_bytes;                   // D part: G dwell groups x PS points x 128 B
  const int stageBytes = lay.stage_bytes;           // [R | R_lo | D_hi | D_lo]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem0);
  uint64_t* full = bars;
  uint64_t* empty = bars + a.n_stage;
  uint64_t* conv = bars + 2 * a.n_stage;
  uint64_t* acc_full = bars + 3 * a.n_stage;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_full + 1);
  const Watch w{a.err, smem_u32(tmem_slot + 1), DEVERR_K_GRAD};

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int s0 = (int)((long long)seg * a.n_slabs / segs), s1 = (int)((long long)(seg + 1) * a.n_slabs / segs);

  if (threadIdx.x == 0) {
    for (int i = 0; i < a.n_stage; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); mbar_init(conv + i, 128); }
    mbar_init(acc_full, 1);
    tmem_slot[1] = 0u;                              // abort flag
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) { tma_prefetch_desc(&tmR); tma_prefetch_desc(&tmD_hi); tma_prefetch_desc(&tmD_lo); }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = __shfl_sync(0xffffffffu, *tmem_slot, 0);   // warp-uniform for the compiler

  if (warp == 0) {
    auto producer = [&]() {
      const uint64_t polD = l2_evict_last(), polR = l2_evict_first();
      int st = 0; uint32_t ph = 0;
      for (int s = s0; s < s1; ++s) {
        GMCO_WAIT(mbar_wait1_addr(w, smem_u32(empty + st), ph ^ 1, DEVERR_W_EMPTY));
        {
          uint8_t* dst = smem + (size_t)st * stageBytes;
          mbar_expect_tx(full + st, (uint32_t)(kRBytes + 2 * dBytes));
          tma_load_3d(&tmR, dst, full + st, 0, s * PS, tile * 4, polR);
          tma_load_3d(&tmD_hi, dst + 2 * kRBytes, full + st, 0, s * PS, 0, polD);
          tma_load_3d(&tmD_lo, dst + 2 * kRBytes + dBytes, full + st, 0, s * PS, 0, polD);
        }
        if (++st == a.n_stage) { st = 0; ph ^= 1; }
      }
    };
    if (elect_one()) producer();                      // one lane issues every TMA load of the CTA
    __syncwarp();
  } else if (warp == 1) {
    auto issuer = [&]() {
      if (s1 <= s0) return;
      // The accumulator is A_pad columns wide; one MMA covers at most 256 of them.  When the columns last (A_pad <= 256)
      // the two correction products go into a separate accumulator at column 256 (see k_dose_tc: the tensor core's
      // accumulate truncates).  Lean issue loop run by ONE elected lane: descriptors differ by 32-bit adds.
      const int n0 = a.A_pad <= 256 ? a.A_pad : 256, n1 = a.A_pad - n0;
      const uint32_t idesc0 = instr_desc(n0, 1, 1), idesc1 = instr_desc(n1 > 0 ? n1 : 16, 1, 1);
      constexpr uint32_t dhi = desc_hi(512, kSwz128Base32);
      const uint32_t corr = a.A_pad <= 256 ? 256u : 0u;
      const int n_stage = a.n_stage;
      const uint32_t base_lo = desc_lo(smem_u32(smem), PS * 128), stage_step = (uint32_t)stageBytes >> 4;
      const uint32_t o_rlo = kRBytes >> 4, o_dhi = (2 * kRBytes) >> 4, o_dlo = (uint32_t)(2 * kRBytes + dBytes) >> 4;
      const uint32_t o_n1 = (8 * PS * 128) >> 4;          // dwell groups 8.. : +8 groups of PS x 128 B
      const uint32_t conv0 = smem_u32(conv), empty0 = smem_u32(empty);
      int st = 0; uint32_t ph = 0;
      for (int s = s0; s < s1; ++s) {
        GMCO_WAIT(mbar_wait1_addr(w, conv0 + 8 * st, ph, DEVERR_W_CONV));
        tc_fence_after();
        {
          const uint32_t r = base_lo + (uint32_t)st * stage_step;
#pragma unroll
          for (int j = 0; j < PS / 8; ++j) {        // K-steps of 8 points = two 4-row swizzle atoms (1024 B)
            const uint32_t rh = r + j * 64, rl = rh + o_rlo, dh = rh + o_dhi, dl = rh + o_dlo;
            const uint32_t first = (s > s0 || j > 0) ? 1u : 0u;
            mma_ss2(tmem, rh, dhi, dh, dhi, idesc0, first);
            mma_ss2(tmem + corr, rh, dhi, dl, dhi, idesc0, corr ? first : 1u);
            mma_ss2(tmem + corr, rl, dhi, dh, dhi, idesc0, 1);
            if (n1 > 0) {
              mma_ss2(tmem + 256, rh, dhi, dh + o_n1, dhi, idesc1, (s > s0 || j > 0) ? 1u : 0u);
              mma_ss2(tmem + 256, rh, dhi, dl + o_n1, dhi, idesc1, 1);
              mma_ss2(tmem + 256, rl, dhi, dh + o_n1, dhi, idesc1, 1);
            }
          }
          tc_commit_addr(empty0 + 8 * st);
          if (s == s1 - 1) tc_commit(acc_full);
        }
        if (++st == n_stage) { st = 0; ph ^= 1; }
      }
    };
    if (elect_one()) issuer();                        // one lane issues every MMA and commit of the CTA
    __syncwarp();
  } else {
    const int q = warp & 3;
    const int L = q * 32 + lane;
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    auto converter_and_epilogue = [&]() {
      // main loop: split each arriving R tile into (hi, lo) in place; element-wise, so the swizzle does not matter
      {
        const int t = threadIdx.x - 64;               // 0..127
        int st = 0; uint32_t ph = 0;
        for (int s = s0; s < s1; ++s) {
          GMCO_WAIT(mbar_wait(w, full + st, ph, DEVERR_W_FULL));
          uint8_t* base = smem + (size_t)st * stageBytes + t * 16;
#pragma unroll
          for (int i = 0; i < kRBytes / 2048; ++i) {
            const float4 v = *reinterpret_cast<const float4*>(base + i * 2048);
            float4 hi, lo;
            hi.x = __uint_as_float(__float_as_uint(v.x) & 0xffffe000u); lo.x = v.x - hi.x;
            hi.y = __uint_as_float(__float_as_uint(v.y) & 0xffffe000u); lo.y = v.y - hi.y;
            hi.z = __uint_as_float(__float_as_uint(v.z) & 0xffffe000u); lo.z = v.z - hi.z;
            hi.w = __uint_as_float(__float_as_uint(v.w) & 0xffffe000u); lo.w = v.w - hi.w;
            *reinterpret_cast<float4*>(base + i * 2048) = hi;
            *reinterpret_cast<float4*>(base + kRBytes + i * 2048) = lo;
          }
          fence_proxy_async();
          mbar_arrive(conv + st);
          if (++st == a.n_stage) { st = 0; ph ^= 1; }
        }
      }
      // Epilogue: thread L owns plan L's row of the tile.  TMEM -> registers -> a padded row in shared memory (the ring is
      // idle by now; pitch A_pad + 4 floats keeps 16 B stores conflict-free) -> ONE bulk asynchronous copy of the whole
      // row (4 A_pad bytes, contiguous in Gpart) per thread.  No cross-thread hand-off: a thread copies what it wrote.
      float* grow = a.Gpart + (((size_t)tile * segs + seg) * 128 + L) * a.A_pad;
      if (s1 > s0) {
        GMCO_WAIT(mbar_wait(w, acc_full, 0, DEVERR_W_ACC_FULL));
        tc_fence_after();
        float* srow = reinterpret_cast<float*>(smem) + (size_t)L * (a.A_pad + 4);
        for (int g = 0; g < G; ++g) {
          uint32_t v[32];
          tmem_ld32(tmem + lane_base + g * 32, v);
          if (a.A_pad <= 256) {
            uint32_t vc[32];
            tmem_ld32(tmem + lane_base + 256 + g * 32, vc);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(vc[j]));
          } else {
            tmem_ld_wait();
          }
#pragma unroll
          for (int i = 0; i < 8; ++i)
            *reinterpret_cast<float4*>(srow + g * 32 + 4 * i) =
                make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]), __uint_as_float(v[4 * i + 2]),
                            __uint_as_float(v[4 * i + 3]));
        }
        fence_proxy_async();
        bulk_store(grow, srow, (uint32_t)a.A_pad * 4u);
        bulk_commit_group();
        bulk_wait_group_read0();                                            // shared memory may go once it has been read
      } else {
        float4* dst = reinterpret_cast<float4*>(grow);
        for (int i = 0; i < a.A_pad / 4; ++i) dst[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    };
    converter_and_epilogue();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { drain_if_aborted(w.abort_addr); tc_fence_after(); tmem_dealloc(tmem, 512); }
}

// ---------------------------------------------------------------------------------------------
// a5 on tensor cores, CTA-PAIR variant (tcgen05 cta_group::2; gmco_options.dose_kernel = 2, off by default: it has not
// run on a GPU).  A stage of k_grad_tc moves 136 KB through shared memory (40 KB landing, 24 KB converter traffic,
// 72 KB read by its six MMAs) in 768 tensor-pipe cycles = 181 B/clk, more than the 128 B/clk an SM's shared memory moves, and its
// 40 KB of operands per stage are 52 B/clk of a measured 57 B/clk from L2 (profiles/r1_tma_bw.md) -- it is bound by
// operand movement, not by the tensor pipe.  Here the two CTAs of a cluster (2, 1, 1) own two adjacent
// plan tiles and the same point slabs.  One MMA spans both: M = 256 plans (each CTA's own R tile is its half of the
// MN-major A operand), N = A_pad dwell positions whose D slab is split between the CTAs by dwell group (each loads
// G / 2 groups of D_hi and of D_lo: its half of the MN-major B operand).  Per stage on C3 a CTA lands 24 KB instead of
// 40 and its shared memory moves 96 KB = 128 B/clk instead of 136 KB (an MMA reads 4 + 4 KB of it instead of 4 + 8);
// the ring holds 6 stages instead of 4.
// Each CTA's TMEM holds the accumulators of its own 128 plans (main at column 0, corrections at column 256).
// Barriers: `full` (own CTA: bytes of its R tile and D halves), `conv` (in the leader: 256 arrivals, the converter
// threads of both CTAs, which have waited for their own `full`), `empty` / `acc_full` (multicast commits).
__host__ __device__ constexpr uint32_t instr_desc_pair_mn(int n) {   // M = 256, both operands MN-major
  return (1u << 4) | (2u << 7) | (2u << 10) | (1u << 15) | (1u << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}

template <int PS>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
k_grad_tc_pair(const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmD_hi,
               const __grid_constant__ CUtensorMap tmD_lo, const GradArgs a) {   // D maps: boxes of G / 2 dwell groups
  if (a.gate && *a.gate == 0) return;                 // both CTAs of a pair take every early exit together
  const int rank = (int)cluster_ctarank();
  const bool leader = rank == 0;
  int seg = blockIdx.y, tile = blockIdx.x, segs = a.segs;   // grid (tiles, segs): a 2-CTA MMA pair is adjacent in x
  if (a.compact_cap && !compact_remap_pair(*a.gate, a.compact_cap, rank, seg, tile, segs)) return;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem0 = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int G = a.A_pad >> 5, Gh = G >> 1;            // dwell groups; this CTA loads groups [rank Gh, rank Gh + Gh)
  const tcl::GradSmem lay = tcl::grad_pair_smem(PS, G, a.n_stage);
  if (!layout_fits(a.err, DEVERR_K_GRAD_PAIR, (uint32_t)(smem0 - smem_raw), lay.end, tcl::grad_tmem_cols(a.A_pad))) return;
  uint8_t* smem = smem0 + lay.ring_off;               // [barriers 1 KB | ring | (epilogue row staging may run past the ring)]
  constexpr int kRBytes = 4 * PS * 128;               // R part: 4 plan groups x PS points x 128 B
  const int dBytes = lay.d_bytes;                     // D part: G / 2 dwell groups x PS points x 128 B
  const int stageBytes = lay.stage_bytes;             // [R | R_lo | D_hi half | D_lo half]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem0);
  uint64_t* full = bars;                              // [n_stage]  in each CTA: its own TMA bytes
  uint64_t* empty = bars + a.n_stage;                 // [n_stage]  in each CTA: multicast commit
  uint64_t* conv = bars + 2 * a.n_stage;              // [n_stage]  used in the leader: 256 arrivals (both CTAs' converters)
  uint64_t* acc_full = bars + 3 * a.n_stage;          //            in each CTA: multicast commit
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_full + 1);
  const Watch w{a.err, smem_u32(tmem_slot + 1), DEVERR_K_GRAD_PAIR};

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int s0 = (int)((long long)seg * a.n_slabs / segs), s1 = (int)((long long)(seg + 1) * a.n_slabs / segs);

  if (threadIdx.x == 0) {
    for (int i = 0; i < a.n_stage; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, 1); mbar_init(conv + i, 256); }
    mbar_init(acc_full, 1);
    tmem_slot[1] = 0u;                                // abort flag
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) { tma_prefetch_desc(&tmR); tma_prefetch_desc(&tmD_hi); tma_prefetch_desc(&tmD_lo); }
  if (warp == 1) tmem_alloc_pair(tmem_slot, 512);
  tc_fence_before();
  cluster_sync_all();                                 // barriers of both CTAs exist before anything arrives on them
  tc_fence_after();
  const uint32_t tmem = __shfl_sync(0xffffffffu, *tmem_slot, 0);

  if (warp == 0) {
    auto producer = [&]() {
      const uint64_t polD = l2_evict_last(), polR = l2_evict_first();
      int st = 0; uint32_t ph = 0;
      for (int s = s0; s < s1; ++s) {
        GMCO_WAIT(mbar_wait1_addr(w, smem_u32(empty + st), ph ^ 1, DEVERR_W_EMPTY));
        {
          uint8_t* dst = smem + (size_t)st * stageBytes;
          mbar_expect_tx(full + st, (uint32_t)(kRBytes + 2 * dBytes));
          tma_load_3d(&tmR, dst, full + st, 0, s * PS, tile * 4, polR);
          tma_load_3d(&tmD_hi, dst + 2 * kRBytes, full + st, 0, s * PS, rank * Gh, polD);
          tma_load_3d(&tmD_lo, dst + 2 * kRBytes + dBytes, full + st, 0, s * PS, rank * Gh, polD);
        }
        if (++st == a.n_stage) { st = 0; ph ^= 1; }
      }
    };
    if (elect_one()) producer();                      // one lane issues every TMA load of the CTA
    __syncwarp();
  } else if (warp == 1) {
    auto issuer = [&]() {                             // run by ONE elected lane of the leader
      if (!leader || s1 <= s0) return;
      const uint32_t idesc = instr_desc_pair_mn(a.A_pad);
      constexpr uint32_t dhi = desc_hi(512, kSwz128Base32);
      const int n_stage = a.n_stage;
      const uint32_t base_lo = desc_lo(smem_u32(smem), PS * 128), stage_step = (uint32_t)stageBytes >> 4;
      const uint32_t o_rlo = kRBytes >> 4, o_dhi = (2 * kRBytes) >> 4, o_dlo = (uint32_t)(2 * kRBytes + dBytes) >> 4;
      const uint32_t empty0 = smem_u32(empty);
      int st = 0; uint32_t ph = 0;
      for (int s = s0; s < s1; ++s) {
        GMCO_WAIT(mbar_wait1_cluster(w, conv + st, ph, DEVERR_W_CONV));
        tc_fence_after();
        const uint32_t r = base_lo + (uint32_t)st * stage_step;
#pragma unroll
        for (int j = 0; j < PS / 8; ++j) {            // K-steps of 8 points = two 4-row swizzle atoms (1024 B)
          const uint32_t rh = r + j * 64, rl = rh + o_rlo, dh = rh + o_dhi, dl = rh + o_dlo;
          const uint32_t first = (s > s0 || j > 0) ? 1u : 0u;
          mma_ss2_pair(tmem, rh, dhi, dh, dhi, idesc, first);
          mma_ss2_pair(tmem + 256, rh, dhi, dl, dhi, idesc, first);
          mma_ss2_pair(tmem + 256, rl, dhi, dh, dhi, idesc, 1);
        }
        tc_commit_pair(empty0 + 8 * st);
        if (s == s1 - 1) tc_commit_pair(smem_u32(acc_full));
        if (++st == n_stage) { st = 0; ph ^= 1; }
      }
    };
    if (elect_one()) issuer();
    __syncwarp();
  } else {
    const int q = warp & 3;
    const int L = q * 32 + lane;
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    auto converter_and_epilogue = [&]() {
      {
        const uint32_t l_conv = leader_addr(conv);
        const int t = threadIdx.x - 64;               // 0..127
        int st = 0; uint32_t ph = 0;
        for (int s = s0; s < s1; ++s) {
          GMCO_WAIT(mbar_wait(w, full + st, ph, DEVERR_W_FULL));   // this CTA's R tile AND its D halves have landed
          uint8_t* base = smem + (size_t)st * stageBytes + t * 16;
#pragma unroll
          for (int i = 0; i < kRBytes / 2048; ++i) {
            const float4 v = *reinterpret_cast<const float4*>(base + i * 2048);
            float4 hi, lo;
            hi.x = __uint_as_float(__float_as_uint(v.x) & 0xffffe000u); lo.x = v.x - hi.x;
            hi.y = __uint_as_float(__float_as_uint(v.y) & 0xffffe000u); lo.y = v.y - hi.y;
            hi.z = __uint_as_float(__float_as_uint(v.z) & 0xffffe000u); lo.z = v.z - hi.z;
            hi.w = __uint_as_float(__float_as_uint(v.w) & 0xffffe000u); lo.w = v.w - hi.w;
            *reinterpret_cast<float4*>(base + i * 2048) = hi;
            *reinterpret_cast<float4*>(base + kRBytes + i * 2048) = lo;
          }
          fence_proxy_async();
          mbar_arrive_cluster(l_conv + 8u * (uint32_t)st);         // releasing arrive at cluster scope
          if (++st == a.n_stage) { st = 0; ph ^= 1; }
        }
      }
      float* grow = a.Gpart + (((size_t)tile * segs + seg) * 128 + L) * a.A_pad;
      if (s1 > s0) {
        GMCO_WAIT(mbar_wait(w, acc_full, 0, DEVERR_W_ACC_FULL));
        tc_fence_after();
        float* srow = reinterpret_cast<float*>(smem) + (size_t)L * (a.A_pad + 4);
        for (int g = 0; g < G; ++g) {
          uint32_t v[32], vc[32];
          tmem_ld32(tmem + lane_base + g * 32, v);
          tmem_ld32(tmem + lane_base + 256 + g * 32, vc);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = __float_as_uint(__uint_as_float(v[j]) + __uint_as_float(vc[j]));
#pragma unroll
          for (int i = 0; i < 8; ++i)
            *reinterpret_cast<float4*>(srow + g * 32 + 4 * i) =
                make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]), __uint_as_float(v[4 * i + 2]),
                            __uint_as_float(v[4 * i + 3]));
        }
        fence_proxy_async();
        bulk_store(grow, srow, (uint32_t)a.A_pad * 4u);
        bulk_commit_group();
        bulk_wait_group_read0();
      } else {
        float4* dst = reinterpret_cast<float4*>(grow);
        for (int i = 0; i < a.A_pad / 4; ++i) dst[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    };
    converter_and_epilogue();
  }
  tc_fence_before();
  if (warp == 1) drain_if_aborted(w.abort_addr);
  cluster_sync_all();                                 // neither CTA's shared memory, TMEM or barriers may go before both are done
  if (warp == 1) { tc_fence_after(); tmem_dealloc_pair(tmem, 512); }
}

// ---------------------------------------------------------------------------------------------
// host side
PFN_cuTensorMapEncodeTiled get_encode() {
  static PFN_cuTensorMapEncodeTiled fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(p);
  }
  return fn;
}

// fp32 matrix [rows][cols] (cols contiguous, cols % 32 == 0) viewed as {32, rows, cols / 32};
// box = {32, box_rows, box_groups}: lands in smem as [group][row][128 B] with the given swizzle.
bool make_map(CUtensorMap* m, const float* base, long long rows, long long cols, int box_rows, int box_groups,
              CUtensorMapSwizzle swz) {
  PFN_cuTensorMapEncodeTiled enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[3] = {32, (cuuint64_t)rows, (cuuint64_t)(cols / 32)};
  cuuint64_t strides[2] = {(cuuint64_t)cols * 4, 128};
  cuuint32_t box[3] = {32, (cuuint32_t)box_rows, (cuuint32_t)box_groups};
  cuuint32_t estr[3] = {1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

struct TcPlan {
  CUtensorMap dose_D_hi, dose_D_lo, dose_T_lo, dose_T;
  CUtensorMap grad_R, grad_D_hi, grad_D_lo;
  CUtensorMap pair_D_hi, pair_D_lo;                // 64-point boxes of the CTA-pair dose kernel
  CUtensorMap gpair_D_hi, gpair_D_lo;              // boxes of G / 2 dwell groups: the CTA-pair gradient kernel
  tcl::Schedule sch{};                             // every size the host chose (tc_layout.h)
  int* tile_seg_dev = nullptr;
  Thresholds thr{};
};

int tc_choose_segs(int n_tiles, int n_pad_points, int num_sms) { return tcl::choose_segs(n_tiles, n_pad_points, num_sms); }

// Opt every tensor kernel in to the full dynamic shared memory once per process.  The attribute is per function and
// process-global: setting it to one handle's exact size would lower the cap under other live handles.
static cudaError_t tc_set_smem_caps() {
  static cudaError_t done = cudaErrorUnknown;
  if (done == cudaSuccess) return done;
  cudaError_t e = cudaFuncSetAttribute(k_dose_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, tcl::kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dose_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, tcl::kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dose_tc<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, tcl::kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dose_tc_pair<4, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, tcl::kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dose_tc_pair<0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, tcl::kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad_tc<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, tcl::kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad_tc_pair<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, tcl::kSmemMax);
  done = e;
  return e;
}

TcPlan* tc_plan_create(const CaseDev& c, const PlanDev& p, const StructHost* sh, int num_sms, int force_single,
                       int wide_accum, int want_grad_pair, cudaStream_t st, char* err, int errlen) {
  if (c.A_pad > kMaxApadTensor) { snprintf(err, errlen, "tensor path supports n_dwell <= 384"); return nullptr; }
  TcPlan* t = new TcPlan();
  t->sch = tcl::choose_schedule(c.A_pad, c.N_pad, p.K_pad, num_sms, force_single, wide_accum, want_grad_pair);
  const tcl::Schedule& q = t->sch;
  if (!q.ok) { snprintf(err, errlen, "shared memory too small for the tensor kernels' rings at this shape"); delete t; return nullptr; }
  for (int s = 0; s < c.S; ++s) { t->thr.d_lo[s] = sh[s].d_lo; t->thr.d_hi[s] = sh[s].d_hi; }
  const int G = q.G;
  const CUtensorMapSwizzle sK = CU_TENSOR_MAP_SWIZZLE_128B, sMN = CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B;
  bool ok = make_map(&t->dose_D_hi, c.D_hi, c.N_alloc, c.A_pad, kPC, 1, sK) &&
            make_map(&t->dose_D_lo, c.D_lo, c.N_alloc, c.A_pad, kPC, 1, sK) &&
            make_map(&t->dose_T, p.T, p.K_pad, c.A_pad, 128, 1, sK) &&
            (q.tlo_resident || (p.T_lo && make_map(&t->dose_T_lo, p.T_lo, p.K_pad, c.A_pad, 128, 1, sK))) &&
            make_map(&t->grad_R, p.R, c.N_alloc, p.K_pad, q.grad_ps, 4, sMN) &&
            make_map(&t->grad_D_hi, c.D_hi, c.N_alloc, c.A_pad, q.grad_ps, G, sMN) &&
            make_map(&t->grad_D_lo, c.D_lo, c.N_alloc, c.A_pad, q.grad_ps, G, sMN);
  if (q.dose_pair)
    ok = ok && make_map(&t->pair_D_hi, c.D_hi, c.N_alloc, c.A_pad, kHalfPC, 2, sK) &&
         make_map(&t->pair_D_lo, c.D_lo, c.N_alloc, c.A_pad, kHalfPC, 2, sK);
  if (q.grad_pair)
    ok = ok && make_map(&t->gpair_D_hi, c.D_hi, c.N_alloc, c.A_pad, q.grad_ps, G / 2, sMN) &&
         make_map(&t->gpair_D_lo, c.D_lo, c.N_alloc, c.A_pad, q.grad_ps, G / 2, sMN);
  if (!ok) { snprintf(err, errlen, "cuTensorMapEncodeTiled failed"); delete t; return nullptr; }
  if (q.tlo_resident) t->dose_T_lo = t->dose_T;   // the resident layout splits T in the kernel; the map is never used for a load
  cudaError_t e = tc_set_smem_caps();
  std::vector<int> seg(q.n_tiles + 1);
  for (int i = 0; i <= q.n_tiles; ++i) seg[i] = i * q.segs;
  t->tile_seg_dev = p.tile_seg;                    // lives in the plan arena; pageable source: staged before the call returns
  if (e == cudaSuccess) e = cudaMemcpyAsync(t->tile_seg_dev, seg.data(), seg.size() * sizeof(int), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) { snprintf(err, errlen, "tensor plan setup: %s", cudaGetErrorString(e)); tc_plan_destroy(t); return nullptr; }
  return t;
}

void tc_plan_destroy(TcPlan* t) {
  if (!t) return;
  delete t;
}

int tc_num_segments(const TcPlan* t) { return t->sch.n_tiles * t->sch.segs; }
int tc_dose_pair(const TcPlan* t) { return t->sch.dose_pair; }
int tc_grad_pair(const TcPlan* t) { return t->sch.grad_pair; }
int tc_dose_kernel(const TcPlan* t) { return t->sch.dose_kernel; }
const int* tc_tile_seg_dev(const TcPlan* t) { return t->tile_seg_dev; }

// at least the static split (a single tile keeps all its CTAs), at most 36 segments: k_step reads one gradient partial
// per segment, two batches of 18 (kernels_lbfgs.cu)
int tc_compact_cap(const TcPlan* t) { return t->sch.segs > 36 ? t->sch.segs : 36; }

// which < 0: both contractions; 0: the dose kernel only; 1: the gradient kernel only (per-kernel timing, gmco_set_profiling)
int launch_tc_eval(const TcPlan* t, const CaseDev& c, const PlanDev& p, float* dose_dbg, const int* gate,
                   int* zero_ctr, int* log_slot, bool compact, int which, cudaStream_t st) {
  const tcl::Schedule& q = t->sch;
  dim3 grid(q.segs, q.n_tiles);
  int n = 0;
  const int cap = compact ? tc_compact_cap(t) : 0;
  if (which != 1) {
    DoseArgs da{};
    da.T = p.T; da.R = p.R; da.Fpart = p.Fpart; da.Weff = compact ? p.WeffC : p.Weff;
    da.compact_cap = cap; da.err = p.dev_err;
    da.tile_struct = c.tile_struct; da.tile_valid = c.tile_valid; da.row_src = c.row_src; da.dose_dbg = dose_dbg;
    da.gate = gate; da.zero_ctr = zero_ctr; da.log_slot = log_slot; da.round_ctr = zero_ctr ? p.rounds_done + 1 : nullptr; da.A_pad = c.A_pad; da.K_pad = p.K_pad; da.K = p.K; da.S = c.S;
    da.n_chunks = q.n_chunks;
    da.segs = q.segs; da.n_stage = q.dose_stages; da.sep_corr = 1;   // T_hi takes at most 256 TMEM columns: both accumulators always fit
    da.n_acc = 1;
    da.tlo_resident = q.tlo_resident; da.thr = t->thr; da.tmem_groups = q.dose_tmem_groups; da.n_main = q.dose_n_main;
    if (q.dose_pair) {
      da.n_stage = q.pair_stages;
      if (q.pair_static) k_dose_tc_pair<4, 6><<<dim3(q.n_tiles, q.segs), kDoseThreads, q.pair_smem, st>>>(t->pair_D_hi, t->pair_D_lo, t->dose_T, da);
      else k_dose_tc_pair<0, 0><<<dim3(q.n_tiles, q.segs), kDoseThreads, q.pair_smem, st>>>(t->pair_D_hi, t->pair_D_lo, t->dose_T, da);
    } else if (q.tlo_resident) k_dose_tc<true><<<grid, kDoseThreads, q.dose_smem, st>>>(t->dose_D_hi, t->dose_D_lo, t->dose_T_lo, t->dose_T, da);
    else if (q.dose_n_main == 2) k_dose_tc<false, true><<<grid, kDoseThreads, q.dose_smem, st>>>(t->dose_D_hi, t->dose_D_lo, t->dose_T_lo, t->dose_T, da);
    else k_dose_tc<false><<<grid, kDoseThreads, q.dose_smem, st>>>(t->dose_D_hi, t->dose_D_lo, t->dose_T_lo, t->dose_T, da);
    if (cudaPeekAtLastError() != cudaSuccess) return -1;   // left for the caller's message
    ++n;
  }
  if (which != 0) {
    GradArgs ga{};
    ga.Gpart = p.Gpart; ga.gate = gate; ga.A_pad = c.A_pad; ga.n_slabs = q.n_slabs; ga.segs = q.segs;
    ga.n_stage = q.grad_stages; ga.compact_cap = cap; ga.err = p.dev_err;
    if (q.grad_pair) {
      ga.n_stage = q.gpair_stages;
      k_grad_tc_pair<16><<<dim3(q.n_tiles, q.segs), kThreads, q.gpair_smem, st>>>(t->grad_R, t->gpair_D_hi, t->gpair_D_lo, ga);
    } else {
      k_grad_tc<16><<<grid, kThreads, q.grad_smem, st>>>(t->grad_R, t->grad_D_hi, t->grad_D_lo, ga);
    }
    if (cudaGetLastError() != cudaSuccess) return -1;
    ++n;
  }
  return n;
}

}  // namespace gmco
