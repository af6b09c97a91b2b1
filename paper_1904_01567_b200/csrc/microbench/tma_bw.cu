// Microbenchmark behind DESIGN.md 5.5: L2 -> SM TMA streaming bandwidth, unicast vs cluster multicast, in the access
// pattern of k_dose_tc.  Not part of libgmco.  Build and run:
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o tma_bw tma_bw.cu -lcuda && ./tma_bw
// Result on B200: profiles/r1_tma_bw.md
// Pattern of
// k_dose_tc: grid (segs, tiles); the `tiles` CTAs of one seg read the same 128-row x 128 B slabs at about the same time.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cudaTypedefs.h>
#include <stdio.h>
#include <stdint.h>
#include <vector>
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory"); }
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok; asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory"); return ok != 0; }
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) { uint32_t s = 0; while (!mbar_try_wait(bar, parity)) if (++s > (1u << 24)) __trap(); }
__device__ __forceinline__ void cluster_sync() { asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
// remote arrive on the same barrier offset of CTA `cta`
__device__ __forceinline__ void mbar_arrive_remote(uint64_t* bar, uint32_t cta) {
  uint32_t ra; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(bar)), "r"(cta));
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(ra) : "memory");
}
constexpr int kStage = 6, kBox = 16384;
// CL = cluster size along y (tiles). Each CTA loads rows/CL of every slab and multicasts to the cluster.
template <int CL>
__global__ void __launch_bounds__(64, 1) k(const __grid_constant__ CUtensorMap tm, int n_chunks, int segs, int G, long long* out) {
  extern __shared__ __align__(1024) uint8_t raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)raw + 1023) & ~(uintptr_t)1023);
  uint64_t* full = (uint64_t*)(smem + kStage * kBox); uint64_t* empty = full + kStage;
  const int seg = blockIdx.x;
  const int c0 = (int)((long long)seg * n_chunks / segs), c1 = (int)((long long)(seg + 1) * n_chunks / segs);
  const uint32_t rank = CL > 1 ? cluster_rank() : 0;
  if (threadIdx.x == 0) { for (int i = 0; i < kStage; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, CL); } asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  if (CL > 1) cluster_sync(); else __syncthreads();
  long long t0 = clock64();
  if (threadIdx.x == 0) {            // producer
    int st = 0; uint32_t ph = 0;
    for (int c = c0; c < c1; ++c) for (int g = 0; g < 2 * G; ++g) {
      mbar_wait(empty + st, ph ^ 1);
      mbar_expect_tx(full + st, kBox);
      uint8_t* dst = smem + st * kBox + rank * (kBox / CL);
      if (CL == 1)
        asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                     ::"r"(smem_u32(dst)), "l"((uint64_t)&tm), "r"(smem_u32(full + st)), "r"(0), "r"(c * 128), "r"(g) : "memory");
      else
        asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%3, %4, %5}], [%2], %6;"
                     ::"r"(smem_u32(dst)), "l"((uint64_t)&tm), "r"(smem_u32(full + st)), "r"(0), "r"(c * 128 + (int)rank * (128 / CL)), "r"(g), "h"((uint16_t)((1 << CL) - 1)) : "memory");
      if (++st == kStage) { st = 0; ph ^= 1; }
    }
  } else if (threadIdx.x == 32) {    // consumer: frees the slot in every CTA of the cluster as soon as the data is there
    int st = 0; uint32_t ph = 0;
    for (int c = c0; c < c1; ++c) for (int g = 0; g < 2 * G; ++g) {
      mbar_wait(full + st, ph);
      if (CL == 1) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(empty + st)) : "memory");
      else for (uint32_t r = 0; r < CL; ++r) mbar_arrive_remote(empty + st, r);
      if (++st == kStage) { st = 0; ph ^= 1; }
    }
  }
  __syncthreads();
  long long t1 = clock64();
  if (CL > 1) cluster_sync();
  if (threadIdx.x == 0) out[blockIdx.y * gridDim.x + blockIdx.x] = t1 - t0;
}
int main() {
  const int N = 12288, A = 512 /* hi and lo as 16 groups of 32 */, segs = 18, tiles = 8, G = 8;
  float* D; cudaMalloc(&D, (size_t)N * A * 4); cudaMemset(D, 0, (size_t)N * A * 4);
  long long* out; cudaMallocManaged(&out, 8 * 160);
  PFN_cuTensorMapEncodeTiled enc; cudaDriverEntryPointQueryResult q;
  cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &q);
  auto mk = [&](int box_rows) { CUtensorMap m; cuuint64_t dims[3] = {32, (cuuint64_t)N, (cuuint64_t)(A / 32)}; cuuint64_t str[2] = {(cuuint64_t)A * 4, 128};
    cuuint32_t box[3] = {32, (cuuint32_t)box_rows, 1}; cuuint32_t es[3] = {1, 1, 1};
    CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, D, dims, str, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r) printf("encode failed %d\n", r); return m; };
  const int smem = kStage * kBox + 1024 + 256;
  auto run = [&](int CL) {
    CUtensorMap m = mk(128 / CL);
    cudaLaunchConfig_t cfg = {}; cfg.gridDim = dim3(segs, tiles); cfg.blockDim = dim3(64); cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1]; at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = CL; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = CL > 1 ? 1 : 0;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e9;
    for (int rep = 0; rep < 5; ++rep) {
      cudaEventRecord(e0);
      cudaError_t e;
      if (CL == 1) { cudaFuncSetAttribute(k<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); e = cudaLaunchKernelEx(&cfg, k<1>, m, N / 128, segs, G, out); }
      else if (CL == 2) { cudaFuncSetAttribute(k<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); e = cudaLaunchKernelEx(&cfg, k<2>, m, N / 128, segs, G, out); }
      else if (CL == 4) { cudaFuncSetAttribute(k<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); e = cudaLaunchKernelEx(&cfg, k<4>, m, N / 128, segs, G, out); }
      else { cudaFuncSetAttribute(k<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); cudaFuncSetAttribute(k<8>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1); e = cudaLaunchKernelEx(&cfg, k<8>, m, N / 128, segs, G, out); }
      cudaEventRecord(e1); cudaError_t e2 = cudaDeviceSynchronize();
      if (e || e2) { printf("CL %d: %s / %s\n", CL, cudaGetErrorString(e), cudaGetErrorString(e2)); return; }
      float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    double cyc = 0; for (int i = 0; i < segs * tiles; ++i) cyc += out[i]; cyc /= segs * tiles;
    const double bytes_per_cta = (double)(N / 128) / segs * 2 * G * kBox;
    printf("CL %d: %.1f us, per CTA %.0f cycles for %.0f KB landed = %.1f B/clk/SM landed; aggregate landed %.2f TB/s\n", CL, best * 1e3, cyc, bytes_per_cta / 1024,
           bytes_per_cta / cyc, bytes_per_cta * segs * tiles / (best * 1e-3) / 1e12);
  };
  for (int CL : {1, 2, 4, 8}) run(CL);
  return 0;
}
