// Microbenchmark behind DESIGN.md 5.1: cycles per tcgen05 kind::tf32 MMA (M = 128, K = 8) for the operand patterns of
// k_dose_tc / k_grad_tc, operands resident (no TMA, no epilogue).  Not part of libgmco.  Build and run:
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o mma_rate mma_rate.cu && ./mma_rate
// Result on B200: profiles/r1_mma_rate.md
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdint.h>
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory"); }
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) { uint32_t s = 0; while (!mbar_try_wait(bar, parity)) if (++s > (1u << 24)) __trap(); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) { asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory"); }
__device__ __forceinline__ void mma_ss(uint32_t d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d), "l"(a), "l"(b), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_ts(uint32_t d, uint32_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d), "r"(a), "l"(b), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo, uint32_t layout) {
  uint64_t d = 0; d |= (uint64_t)((saddr >> 4) & 0x3fff); d |= (uint64_t)((lbo >> 4) & 0x3fff) << 16; d |= (uint64_t)((sbo >> 4) & 0x3fff) << 32;
  d |= (uint64_t)1 << 46; d |= (uint64_t)layout << 61; return d;
}
__host__ __device__ constexpr uint32_t instr_desc(int n, int amn, int bmn) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)amn << 15) | ((uint32_t)bmn << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
// mode 0: TS N=64 | 1: dose pattern (TS,TS,SS) N=64 | 2: SS N=64 K-major | 3: SS N=256 MN-major (grad) | 4: TS N=128 | 5: TS N=256
// 6: dose pattern with N=128 | 7: SS N=128 K-major | 8: (TS,TS) only N=64, two accumulators
__global__ void __launch_bounds__(128, 1) k(int mode, int iters, long long* out) {
  extern __shared__ __align__(1024) uint8_t raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)raw + 1023) & ~(uintptr_t)1023);
  __shared__ uint64_t bar; __shared__ uint32_t slot;
  const int warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < 160 * 1024 / 4; i += 128) ((float*)smem)[i] = 1e-3f * (i & 255);
  if (threadIdx.x == 0) { mbar_init(&bar, 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  if (warp == 0) { asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&slot)) : "memory");
                   asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory"); }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); __syncthreads(); asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = slot;
  if (threadIdx.x == 0) {
    const uint32_t base = smem_u32(smem);
    long long t0 = clock64();
    int n_mma = 0;
    for (int it = 0; it < iters; ++it) {
      // one "stage": distinct smem per stage slot like the ring (6 slots of 16 KB at offset 32 KB.., A_lo at 0..)
      const uint32_t sb = base + 32768 + (it % 6) * 16384;
      const uint32_t acc = 256 + (it & 1) * 128;
      if (mode == 0 || mode == 4 || mode == 5) {
        const int N = mode == 0 ? 64 : mode == 4 ? 128 : 256;
        const uint32_t id = instr_desc(N, 0, 0);
        for (int j = 0; j < 4; ++j) for (int r = 0; r < 3; ++r) { mma_ts(mode == 5 ? 256 + tmem : tmem + acc + (mode == 0 ? (r & 1) * 64 : 0), tmem + (it % 8) * 32 + j * 8, smem_desc(sb + (r & 1) * 8192, 16, 1024, 2) + 2 * j, id, 1); ++n_mma; }
      } else if (mode == 1 || mode == 6) {
        const int N = mode == 1 ? 64 : 128;
        const uint32_t id = instr_desc(N, 0, 0);
        const uint32_t accm = mode == 1 ? tmem + acc : tmem + 256, accc = mode == 1 ? tmem + acc + 64 : tmem + 384;
        const uint64_t alo = smem_desc(base + (it % 2) * 16384, 16, 1024, 2);
        for (int j = 0; j < 4; ++j) {
          mma_ts(accm, tmem + (it % 8) * 32 + j * 8, smem_desc(sb, 16, 1024, 2) + 2 * j, id, 1);
          mma_ts(accc, tmem + (it % 8) * 32 + j * 8, smem_desc(sb + 8192, 16, 1024, 2) + 2 * j, id, 1);
          mma_ss(accc, alo + 2 * j, smem_desc(sb, 16, 1024, 2) + 2 * j, id, 1);
          n_mma += 3;
        }
      } else if (mode == 2 || mode == 7) {
        const int N = mode == 2 ? 64 : 128;
        const uint32_t id = instr_desc(N, 0, 0);
        const uint64_t alo = smem_desc(base + (it % 2) * 16384, 16, 1024, 2);
        for (int j = 0; j < 4; ++j) for (int r = 0; r < 3; ++r) { mma_ss(tmem + acc + (mode == 2 ? (r & 1) * 64 : 0), alo + 2 * j, smem_desc(sb + (r & 1) * 8192, 16, 1024, 2) + 2 * j, id, 1); ++n_mma; }
      } else if (mode == 3) {
        const uint32_t id = instr_desc(256, 1, 1);
        const int PS = 32;
        const uint32_t st = base + (it % 2) * 98304 / 2;   // just two regions
        for (int j = 0; j < 4; ++j) {
          const uint64_t rhi = smem_desc(st + j * 1024, PS * 128, 512, 1), rlo = smem_desc(st + 16384 + j * 1024, PS * 128, 512, 1);
          const uint64_t dhi = smem_desc(base + 65536 + j * 1024, PS * 128, 512, 1), dlo = smem_desc(base + 65536 + 32768 + j * 1024, PS * 128, 512, 1);
          mma_ss(tmem, rhi, dhi, id, 1); mma_ss(tmem + 256, rhi, dlo, id, 1); mma_ss(tmem + 256, rlo, dhi, id, 1);
          n_mma += 3;
        }
      } else if (mode == 8) {
        const uint32_t id = instr_desc(64, 0, 0);
        for (int j = 0; j < 4; ++j) {
          mma_ts(tmem + acc, tmem + (it % 8) * 32 + j * 8, smem_desc(sb, 16, 1024, 2) + 2 * j, id, 1);
          mma_ts(tmem + acc + 64, tmem + (it % 8) * 32 + j * 8, smem_desc(sb + 8192, 16, 1024, 2) + 2 * j, id, 1);
          n_mma += 2;
        }
      }
    }
    tc_commit(&bar);
    mbar_wait(&bar, 0);
    long long t1 = clock64();
    if (blockIdx.x == 0) { out[0] = t1 - t0; out[1] = n_mma; }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); __syncthreads();
  if (warp == 0) { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory"); }
}
int main() {
  long long* out; cudaMallocManaged(&out, 16);
  cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  const char* names[] = {"TS N=64", "dose pattern TS,TS,SS N=64", "SS N=64", "grad SS N=256 MN-major", "TS N=128", "TS N=256", "dose pattern N=128", "SS N=128", "TS,TS N=64"};
  for (int grid : {1, 148}) for (int mode = 0; mode < 9; ++mode) {
    for (int rep = 0; rep < 2; ++rep) { k<<<grid, 128, 200 * 1024>>>(mode, 2000, out); cudaError_t e = cudaDeviceSynchronize(); if (e) { printf("mode %d: %s\n", mode, cudaGetErrorString(e)); return 1; } }
    const int N = (mode == 3 || mode == 5) ? 256 : (mode == 4 || mode == 6 || mode == 7) ? 128 : 64;
    printf("grid %3d mode %d %-28s cycles/MMA %.1f  (floor %d)\n", grid, mode, names[mode], (double)out[0] / out[1], N / 2);
  }
  return 0;
}
