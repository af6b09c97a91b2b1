// tc_layout.h -- shared-memory / TMEM carve-up and launch schedule of the tensor kernels (kernels_tc.cu).
//
// Plain C++ (no CUDA types): the kernels take their offsets from these functions, tc_plan_create takes its
// sizes from them, and gmco_tc_info (include/gmco.h) reports them, so that `-m "not gpu"` tests can prove on
// the CPU that for every shape the host can choose the carve-up fits the launched dynamic shared memory, the
// TMEM columns stay within 512 and the TMA boxes stay inside the allocations (tests/test_tc_layout_model.py).
// Product code; shares nothing with oracle/.
#pragma once

#include <stdint.h>

#if defined(__CUDACC__)
#define GMCO_HD __host__ __device__ __forceinline__
#else
#define GMCO_HD inline
#endif

namespace gmco {
namespace tcl {

constexpr int kPC = 128;                   // points per dose chunk = MMA N of the dose contraction
constexpr int kSlabBytes = kPC * 128;      // one 32-dwell slab of a dose chunk, one part (hi or lo): 16 KB
constexpr int kTloBox = 128 * 128;         // T_lo: 128 plans x 32 dwell: 16 KB
constexpr int kTmemGroups = 8;             // dwell groups of T_hi kept in TMEM (256 columns)
constexpr int kTmemGroupsSplit = 4;        // the same with the split main accumulator of the streamed layout (128 columns)
constexpr int kTmemCols = 512;             // TMEM columns of one SM
constexpr int kScratchBytes = 8 * 4096;    // T_hi transposition scratch (streamed layout), one 4 KB slab per epilogue warp
constexpr int kHalfPC = kPC / 2;
constexpr int kHalfSlab = kHalfPC * 128;   // 8 KB: 64 points x 32 dwell of one part
constexpr int kPairEntry = 2 * kHalfSlab;  // ring entry of the CTA-pair kernel: two dwell groups of a half slab
constexpr int kMaxGroups = 12;             // kMaxApadTensor / 32
constexpr int kSmemMax = 227 * 1024;       // opt-in dynamic shared memory per CTA on sm_100
constexpr int kAlign = 1024;               // SWIZZLE_128B operands need 1024 B alignment; the base is aligned up by hand
constexpr int kBarBytes = 512;             // barrier block of the dose kernels
constexpr int kGradBarBytes = 1024;        // barrier block of the gradient kernel (in front of its ring)
constexpr int kDoseMaxStages = 12, kGradMaxStages = 9;

// ---- k_dose_tc<resident> ------------------------------------------------------------------------------------------
struct DoseSmem {
  int tlo_bytes;      // resident: T_lo [G][128][128 B]; streamed: T_hi tail [G - kTmemGroups][128][128 B]
  int stage_bytes;    // ring entry: D slab (+ the streamed T_lo slab behind a D_hi slab)
  int ring_off, ring_bytes;
  int scratch_off;    // streamed layout: the last kScratchBytes of the ring double as the prologue's scratch
  int scr_slot;       // first ring slot that overlaps the scratch
  int bars_off;       // uint64 barriers: full[n], empty[n], tg_ready[kMaxGroups], tin_full[kMaxGroups], acc_full[2], acc_empty[2]
  int n_bars;
  int slot_off;       // uint32 TMEM base address, uint32 abort flag
  int end;            // bytes used from the aligned base
};
// tmem_groups: dwell groups of T_hi that live in TMEM (kTmemGroups, or kTmemGroupsSplit for the split-main layout)
GMCO_HD DoseSmem dose_smem(bool resident, int G, int n_stage, int tmem_groups = kTmemGroups) {
  DoseSmem s;
  const int Gs = resident ? 0 : (G > tmem_groups ? G - tmem_groups : 0);
  s.tlo_bytes = (resident ? G : Gs) * kTloBox;
  s.stage_bytes = resident ? kSlabBytes : kSlabBytes + kTloBox;
  s.ring_off = s.tlo_bytes;
  s.ring_bytes = n_stage * s.stage_bytes;
  s.scratch_off = s.ring_off + s.ring_bytes - kScratchBytes;
  s.scr_slot = (s.ring_bytes - kScratchBytes) / s.stage_bytes;
  s.bars_off = s.ring_off + s.ring_bytes;
  s.n_bars = 2 * n_stage + 2 * kMaxGroups + 4;
  s.slot_off = s.bars_off + 8 * s.n_bars;
  s.end = s.slot_off + 8;
  return s;
}
// TMEM columns: T_hi of min(G, tmem_groups) groups, then one accumulator buffer: n_main main accumulators (the main
// product's adds split by dwell-group block) + the separate correction accumulator, 128 points each
GMCO_HD int dose_tmem_acc_col(int G, int tmem_groups = kTmemGroups) { return (G < tmem_groups ? G : tmem_groups) * 32; }
GMCO_HD int dose_tmem_cols(int G, int tmem_groups = kTmemGroups, int n_main = 1) {
  return dose_tmem_acc_col(G, tmem_groups) + (n_main + 1) * kPC;
}

// ---- k_dose_tc_pair ---------------------------------------------------------------------------------------------------
struct PairSmem {
  int tlo_bytes, ring_off, ring_bytes, bars_off, n_bars, slot_off, end;
};
GMCO_HD PairSmem pair_smem(int G, int n_stage) {
  PairSmem s;
  s.tlo_bytes = G * kTloBox;
  s.ring_off = s.tlo_bytes;
  s.ring_bytes = n_stage * kPairEntry;
  s.bars_off = s.ring_off + s.ring_bytes;
  s.n_bars = 2 * n_stage + 2 * kTmemGroups + 4;   // full[n], empty[n], tg_ready[8], tin_full[8], acc_full[2], acc_empty[2]
  s.slot_off = s.bars_off + 8 * s.n_bars;
  s.end = s.slot_off + 8;
  return s;
}
GMCO_HD int pair_tmem_cols(int G) { return G * 32 + 2 * kPC; }   // T_hi + two accumulator buffers

// ---- k_grad_tc<PS> ----------------------------------------------------------------------------------------------------
struct GradSmem {
  int r_bytes, d_bytes, stage_bytes;   // stage = [R | R_lo | D_hi | D_lo]
  int ring_off, ring_bytes;
  int n_bars;                          // full[n], empty[n], conv[n], acc_full; then the TMEM slot and the abort flag
  int staging_bytes;                   // epilogue: one padded accumulator row per plan, laid over the idle ring
  int end;
};
GMCO_HD GradSmem grad_smem(int PS, int G, int n_stage) {
  GradSmem s;
  s.r_bytes = 4 * PS * 128;
  s.d_bytes = G * PS * 128;
  s.stage_bytes = 2 * s.r_bytes + 2 * s.d_bytes;
  s.ring_off = kGradBarBytes;
  s.ring_bytes = n_stage * s.stage_bytes;
  s.n_bars = 3 * n_stage + 1;
  s.staging_bytes = 128 * (G * 32 + 4) * 4;
  s.end = s.ring_off + (s.ring_bytes > s.staging_bytes ? s.ring_bytes : s.staging_bytes);
  return s;
}
GMCO_HD int grad_tmem_cols(int A_pad) { return A_pad <= 256 ? 256 + A_pad : A_pad; }

// ---- k_grad_tc_pair<PS> (gmco_options.dose_kernel = 2; at most 256 dwell positions, even tile and group counts) ------
// Two CTAs of a cluster own two adjacent plan tiles and the same point slabs; each loads its own R tile and HALF of the
// dwell groups of every D slab, so a stage is [R | R_lo | D_hi half | D_lo half].
GMCO_HD GradSmem grad_pair_smem(int PS, int G, int n_stage) {
  GradSmem s;
  s.r_bytes = 4 * PS * 128;
  s.d_bytes = (G / 2) * PS * 128;
  s.stage_bytes = 2 * s.r_bytes + 2 * s.d_bytes;
  s.ring_off = kGradBarBytes;
  s.ring_bytes = n_stage * s.stage_bytes;
  s.n_bars = 3 * n_stage + 1;
  s.staging_bytes = 128 * (G * 32 + 4) * 4;
  s.end = s.ring_off + (s.ring_bytes > s.staging_bytes ? s.ring_bytes : s.staging_bytes);
  return s;
}

// ---- host-side schedule -------------------------------------------------------------------------------------------------
// Point segments per plan tile.  Up to num_sms / n_tiles the grid is one wave of CTAs.  With many tiles one wave leaves
// SMs idle (79 tiles of a 10 000-plan pool: 79 of 148) or unevenly loaded (C4: 32 tiles x 4 = 128 CTAs), so the grid
// may run to several waves of shorter CTAs when this model says it pays: time ~ waves x (chunks per CTA + 1), the
// "+ 1" standing for a CTA's prologue and tail (about one 128-point chunk's worth).
inline int choose_segs(int n_tiles, int n_pad_points, int num_sms) {
  const int n_chunks = (n_pad_points + kPC - 1) / kPC;
  auto cost = [&](int s) {
    const int waves = (n_tiles * s + num_sms - 1) / num_sms;
    return waves * ((n_chunks + s - 1) / s + 1);
  };
  const int s0 = num_sms / n_tiles > 0 ? num_sms / n_tiles : 1;
  int best = s0;
  for (int s = s0 + 1; s <= 36 && s <= n_chunks; ++s)
    if (cost(s) < cost(best) && 100 * cost(s) < 95 * cost(s0)) best = s;
  return best;
}

enum DoseKernelId { kDoseResident = 0, kDoseStreamed = 1, kDosePairStatic = 2, kDosePairRing = 3 };

struct Schedule {
  int ok;                  // 0: the shape does not fit the tensor route
  int G, n_tiles, segs, n_chunks;
  int tlo_resident, dose_stages, dose_smem;
  int dose_tmem_groups, dose_n_main;   // streamed layout only: 4 groups of T_hi in TMEM and two main accumulators when wide_accum is on
  int dose_pair, pair_static, pair_stages, pair_smem;
  int grad_ps, grad_stages, grad_smem, n_slabs;
  int grad_pair, gpair_stages, gpair_smem;   // CTA-pair gradient kernel (option): ring depth and launched bytes
  int dose_kernel;         // DoseKernelId of the kernel that launch_tc_eval dispatches
};

// Every size the host chooses for a case of A_pad dwell columns, N_pad padded points and K_pad padded plans.
// force_single != 0 keeps the single-CTA dose kernel where the CTA-pair kernel would be eligible.  wide_accum != 0
// selects the split-main layout for the streamed dose kernel (more than 256 dwell positions).
// want_grad_pair != 0 (gmco_options.dose_kernel = 2) also runs the gradient contraction on CTA pairs where the shape allows.
inline Schedule choose_schedule(int A_pad, int N_pad, int K_pad, int num_sms, int force_single, int wide_accum = 0,
                                int want_grad_pair = 0) {
  Schedule t{};
  t.G = A_pad / 32;
  t.n_tiles = K_pad / 128;
  if (A_pad < 32 || A_pad % 32 || t.G > kMaxGroups || t.n_tiles < 1 || N_pad < 1 || num_sms < 1) return t;
  const int G = t.G;
  t.segs = choose_segs(t.n_tiles, N_pad, num_sms);
  t.n_chunks = (N_pad + kPC - 1) / kPC;
  const int slack = kAlign + kBarBytes;
  // dose kernel: T_lo resident when it leaves room for >= 4 ring stages, else streamed with every D_hi slab
  t.tlo_resident = (G <= kTmemGroups && G * kTloBox + 4 * kSlabBytes + slack <= kSmemMax) ? 1 : 0;
  t.dose_tmem_groups = (!t.tlo_resident && wide_accum) ? kTmemGroupsSplit : kTmemGroups;
  t.dose_n_main = (!t.tlo_resident && wide_accum) ? 2 : 1;
  {
    const DoseSmem probe = dose_smem(t.tlo_resident != 0, G, 0, t.dose_tmem_groups);
    const int fixed = probe.tlo_bytes + slack;
    t.dose_stages = (kSmemMax - fixed) / probe.stage_bytes;
    if (t.dose_stages > kDoseMaxStages) t.dose_stages = kDoseMaxStages;
    if (t.dose_stages < 2 || t.dose_stages * probe.stage_bytes < kScratchBytes) return t;
    t.dose_smem = fixed + t.dose_stages * probe.stage_bytes;
  }
  // gradient kernel: 16-point stages (the ring is deeper in stages than with 32: measured faster)
  t.grad_ps = 16;
  {
    const GradSmem probe = grad_smem(t.grad_ps, G, 0);
    t.grad_stages = (kSmemMax - 2 * kGradBarBytes) / probe.stage_bytes;
    if (t.grad_stages > kGradMaxStages) t.grad_stages = kGradMaxStages;
    if (t.grad_stages < 2) return t;
    t.grad_smem = kAlign + grad_smem(t.grad_ps, G, t.grad_stages).end;
    t.n_slabs = N_pad / t.grad_ps;
  }
  // CTA-pair dose kernel: resident layout and an even number of plan tiles.  With an odd number of dwell groups the last
  // ring entry of a pass is half empty (the TMA box's second group lies outside the tensor and is zero-filled; its MMAs
  // are skipped): executed against the oracle on the CPU emulation for G = 1, 3, 5, 7 (tests/test_emu_kernels.py); the
  // GPU parity test of that path is tests/test_gpu_zz_pair.py.
  t.dose_pair = (t.tlo_resident && t.n_tiles % 2 == 0 && !force_single) ? 1 : 0;
  if (t.dose_pair) {
    const int fixedp = G * kTloBox + slack;
    t.pair_stages = (kSmemMax - fixedp) / kPairEntry;
    if (t.pair_stages > kDoseMaxStages) t.pair_stages = kDoseMaxStages;
    t.pair_smem = fixedp + t.pair_stages * kPairEntry;
    // static issue schedule for the production shape (A_pad 193..256: 12 entries per chunk, ring of 6)
    t.pair_static = ((G + 1) / 2 == 4 && t.pair_stages >= 6) ? 1 : 0;
    if (t.pair_static) { t.pair_stages = 6; t.pair_smem = fixedp + 6 * kPairEntry; }
  }
  // CTA-pair gradient kernel: the split of D over the pair is by dwell group, so their number must be even; the
  // accumulator pair (main + corrections) needs A_pad <= 256; the CTA split must be the dose kernel's (k_step reads both)
  t.grad_pair = (want_grad_pair && t.dose_pair && G % 2 == 0 && A_pad <= 256) ? 1 : 0;
  if (t.grad_pair) {
    const GradSmem probe = grad_pair_smem(t.grad_ps, G, 0);
    t.gpair_stages = (kSmemMax - 2 * kGradBarBytes) / probe.stage_bytes;
    if (t.gpair_stages > kGradMaxStages) t.gpair_stages = kGradMaxStages;
    if (t.gpair_stages < 2) t.grad_pair = 0;
    else t.gpair_smem = kAlign + grad_pair_smem(t.grad_ps, G, t.gpair_stages).end;
  }
  t.dose_kernel = t.dose_pair ? (t.pair_static ? kDosePairStatic : kDosePairRing)
                              : (t.tlo_resident ? kDoseResident : kDoseStreamed);
  t.ok = 1;
  return t;
}

}  // namespace tcl
}  // namespace gmco
