// emu_ptx.h -- TEST INFRASTRUCTURE ONLY: a software model of the PTX instructions that csrc/gmco_ptx.cuh issues.
//
// tests/emu/build_emu.py compiles the kernels with `#include "gmco_ptx.cuh"` redirected to this file: same function
// names and signatures, each implemented on the emulation runtime (emu_runtime.cc) instead of inline assembly:
//   mbarrier        phase / pending-arrival / tx-count state machine, kept beside (not in) the 8 bytes it names
//   TMA             tiled copies through an emulated tensor map: box, out-of-bounds zero fill, 128 B swizzles, complete_tx
//   tcgen05         TMEM as a 128 x 512 array per CTA, alloc / dealloc bookkeeping, MMA decoded from the instruction and
//                   shared-memory descriptors (K-major SWIZZLE_128B, MN-major SWIZZLE_128B_BASE32B), tf32 operands,
//                   truncating fp32 accumulate, commit -> mbarrier arrive, 32x32b ld / st with the lane-quadrant rule
//   clusters        rank, mapa, cluster barrier, cta_group::2 forms (M = 256 over two CTAs, multicast commit)
// Every address the "hardware" touches is checked against the CTA's shared-memory window, the TMEM allocation and the
// device allocations; a violation is recorded (emu_violations()) instead of raising anything.
#pragma once

#include "emu_core.h"

namespace emu {
uint32_t smem_window_addr(const void* p);                 // generic pointer into shared memory -> shared::cta window address
void mbar_init(uint32_t addr, uint32_t count);
void mbar_arrive(uint32_t addr, uint32_t tx_bytes);       // one arrival (+ expect_tx when tx_bytes > 0); addr may be shared::cluster
bool mbar_try_wait(uint32_t addr, uint32_t parity);
uint32_t ld_shared_u32(uint32_t addr);
void st_shared_u32(uint32_t addr, uint32_t v);
uint32_t dynamic_smem_bytes();
bool elect_one_sync();
void tma_load(const CUtensorMap* map, uint32_t dst, uint32_t bar, int c0, int c1, int c2, bool pair);
void tmem_alloc(uint32_t dst_addr, uint32_t ncols, bool pair);
void tmem_dealloc(uint32_t taddr, uint32_t ncols, bool pair);
void tc_commit(uint32_t bar, bool pair);
void tc_mma(uint32_t d_tmem, bool a_in_tmem, uint32_t a_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc, bool pair);
void tmem_ld32(uint32_t taddr, uint32_t* v);
void tmem_st32(uint32_t taddr, const uint32_t* v);
uint32_t cluster_rank();
void cluster_barrier();
uint32_t map_to_rank(uint32_t addr, uint32_t rank);
void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar);
void bulk_s2g(void* dst, uint32_t src, uint32_t bytes);
void bulk_wait_read();
}  // namespace emu

namespace gmco {

inline uint32_t smem_u32(const void* p) { return emu::smem_window_addr(p); }

inline void mbar_init(uint64_t* bar, uint32_t count) { emu::mbar_init(smem_u32(bar), count); }
inline void mbar_expect_tx(uint64_t* bar, uint32_t bytes) { emu::mbar_arrive(smem_u32(bar), bytes); }
inline void mbar_arrive(uint64_t* bar) { emu::mbar_arrive(smem_u32(bar), 0); }
inline bool mbar_try_wait_addr(uint32_t bar, uint32_t parity) { return emu::mbar_try_wait(bar, parity); }
inline bool mbar_try_wait_cluster_addr(uint32_t bar, uint32_t parity) { return emu::mbar_try_wait(bar, parity); }

inline unsigned long long global_ns() { return emu::virtual_ns(); }
inline uint32_t ld_flag(uint32_t addr) { return emu::ld_shared_u32(addr); }
inline void st_flag(uint32_t addr, uint32_t v) { emu::st_shared_u32(addr, v); }
inline uint32_t dynamic_smem_size() { return emu::dynamic_smem_bytes(); }
inline bool elect_one() { return emu::elect_one_sync(); }
inline void fence_barrier_init() {}

inline uint64_t l2_evict_last() { return 1; }
inline uint64_t l2_evict_first() { return 2; }
inline uint64_t l2_evict_normal() { return 3; }
inline void tma_load_3d(const CUtensorMap* map, void* dst, uint64_t* bar, int c0, int c1, int c2, uint64_t) {
  emu::tma_load(map, smem_u32(dst), smem_u32(bar), c0, c1, c2, false);
}
inline void tma_prefetch_desc(const CUtensorMap*) {}

inline void tc_fence_before() {}
inline void tc_fence_after() {}
inline void tmem_alloc(uint32_t* dst_smem, uint32_t ncols) { emu::tmem_alloc(smem_u32(dst_smem), ncols, false); }
inline void tmem_dealloc(uint32_t taddr, uint32_t ncols) { emu::tmem_dealloc(taddr, ncols, false); }
inline void tc_commit(uint64_t* bar) { emu::tc_commit(smem_u32(bar), false); }
inline void tc_commit_addr(uint32_t bar) { emu::tc_commit(bar, false); }
inline void mma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
  emu::tc_mma(d_tmem, false, 0, a_desc, b_desc, idesc, acc, false);
}
inline void mma_ts2(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t acc) {
  emu::tc_mma(d_tmem, true, a_tmem, 0, ((uint64_t)b_hi << 32) | b_lo, idesc, acc, false);
}
inline void mma_ss2(uint32_t d_tmem, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t acc) {
  emu::tc_mma(d_tmem, false, 0, ((uint64_t)a_hi << 32) | a_lo, ((uint64_t)b_hi << 32) | b_lo, idesc, acc, false);
}
inline void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) { emu::tmem_ld32(taddr, v); }
inline void tmem_ld_wait() {}
inline void tmem_st32(uint32_t taddr, const uint32_t (&v)[32]) { emu::tmem_st32(taddr, v); }
inline void tmem_st_wait() {}

// cvt.rna.tf32.f32: round to nearest, ties away from zero, to a 10-bit mantissa
inline float tf32_rn(float v) {
  uint32_t u = __float_as_uint(v);
  if ((u & 0x7f800000u) == 0x7f800000u) return v;          // inf / nan
  u = (u + 0x1000u) & 0xffffe000u;
  return __uint_as_float(u);
}
inline void fence_proxy_async() {}

inline uint32_t cluster_ctarank() { return emu::cluster_rank(); }
inline void cluster_sync_all() { emu::cluster_barrier(); }
inline uint32_t leader_addr(const void* p) { return emu::map_to_rank(smem_u32(p), 0); }
inline void mbar_arrive_cluster(uint32_t cluster_bar) { emu::mbar_arrive(cluster_bar, 0); }
inline void tma_load_3d_pair(const CUtensorMap* map, void* dst, uint32_t leader_bar, int c0, int c1, int c2, uint64_t) {
  emu::tma_load(map, smem_u32(dst), leader_bar, c0, c1, c2, true);
}
inline void tmem_alloc_pair(uint32_t* dst_smem, uint32_t ncols) { emu::tmem_alloc(smem_u32(dst_smem), ncols, true); }
inline void tmem_dealloc_pair(uint32_t taddr, uint32_t ncols) { emu::tmem_dealloc(taddr, ncols, true); }
inline void tc_commit_pair(uint32_t bar) { emu::tc_commit(bar, true); }
inline void mma_ts2_pair(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t acc) {
  emu::tc_mma(d_tmem, true, a_tmem, 0, ((uint64_t)b_hi << 32) | b_lo, idesc, acc, true);
}
inline void mma_ss2_pair(uint32_t d_tmem, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t acc) {
  emu::tc_mma(d_tmem, false, 0, ((uint64_t)a_hi << 32) | a_lo, ((uint64_t)b_hi << 32) | b_lo, idesc, acc, true);
}

inline void bulk_load(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar) {
  emu::bulk_g2s(smem_u32(dst_smem), src, bytes, smem_u32(bar));
}
inline void bulk_store(void* dst, const void* src_smem, uint32_t bytes) { emu::bulk_s2g(dst, smem_u32(src_smem), bytes); }
inline void bulk_commit_group() {}
inline void bulk_wait_group_read0() { emu::bulk_wait_read(); }

}  // namespace gmco
