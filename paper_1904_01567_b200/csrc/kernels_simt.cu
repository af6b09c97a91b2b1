// kernels_simt.cu -- case setup and the plain-fp32 (CUDA-core) evaluation kernels.
//
// These kernels are (1) the GMCO_PREC_SIMT_FP32 route of the two contractions, (2) the final
// dose pass of gmco_result that produces objective terms and DVH indices (a8), and (3) the only
// route that can hand dose to the caller (gmco_evaluate's debug output).  The production
// contraction is the tcgen05 kernel in kernel_fused_tc.cu.
#include "gmco_internal.cuh"
#include "gmco_ptx.cuh"
#include "penalty.cuh"

namespace gmco {

// ---------------------------------------------------------------------------------------------
// a0: D_user [N][ldD] -> D [N_alloc][A_pad] (rows regrouped/padded via row_src), optional tf32 parts.
__global__ void k_pad_D(const float* __restrict__ Du, long long ldD, int A, const int* __restrict__ row_src,
                        int N_alloc, int A_pad, float* __restrict__ D, float* __restrict__ D_hi,
                        float* __restrict__ D_lo) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)N_alloc * A_pad) return;
  const int r = (int)(idx / A_pad), a = (int)(idx % A_pad);
  const int src = row_src[r];
  const float v = (src >= 0 && a < A) ? Du[(long long)src * ldD + a] : 0.f;
  D[idx] = v;
  if (D_hi) {
    const float hi = tf32_rn(v);
    D_hi[idx] = hi;
    D_lo[idx] = tf32_rn(v - hi);
  }
}

int launch_setup_case(const CaseDev& c, const float* D_user, long long ldD, const int* row_src_dev,
                      bool want_split, cudaStream_t st) {
  const long long tot = (long long)c.N_alloc * c.A_pad;
  k_pad_D<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(D_user, ldD, c.A, row_src_dev, c.N_alloc, c.A_pad, c.D,
                                                          want_split ? c.D_hi : nullptr, want_split ? c.D_lo : nullptr);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------
// a2-a4 (SIMT): one 64-point x 64-plan tile per CTA, 16x16 threads, 4x4 outputs each.
//   d = D t (Eq. 1), penalty + derivative (Eq. 2), per-tile objective partials (Eq. 4).
// Fpart [tile_p][K_pad][2] holds the (lo, hi) sums of this tile's points; tiles are uniform in
// structure, so summing the tiles of one structure gives the objective terms as well.
template <bool WRITE_R, bool DVH>
__global__ void __launch_bounds__(256)
k_simt_dose(const float* __restrict__ D, const float* __restrict__ T, int A_pad, int N_alloc, int K_pad, int K, int S,
            const float* __restrict__ pt_lo, const float* __restrict__ pt_hi, const int* __restrict__ tile_struct,
            const float* __restrict__ Weff, float* __restrict__ Fpart, float* __restrict__ R,
            float* __restrict__ dose_out, const int* __restrict__ row_src,
            const float* __restrict__ dvh_thr, int* __restrict__ cnt, const int* __restrict__ sel_pos,
            float* __restrict__ sel_buf, int n_sel, const int* __restrict__ gate) {
  if (gate && *gate == 0) return;
  __shared__ float Ds[16][68];
  __shared__ float Ts[16][68];
  __shared__ float red[16][64][2];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int p0 = blockIdx.x * 64, k0 = blockIdx.y * 64;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  const int lr = tid >> 2, lc = (tid & 3) * 4;       // loader: row 0..63, 4 consecutive k
  for (int a0 = 0; a0 < A_pad; a0 += 16) {
    const float4 dv = *reinterpret_cast<const float4*>(D + (long long)(p0 + lr) * A_pad + a0 + lc);
    const float4 tv = *reinterpret_cast<const float4*>(T + (long long)(k0 + lr) * A_pad + a0 + lc);
    Ds[lc + 0][lr] = dv.x; Ds[lc + 1][lr] = dv.y; Ds[lc + 2][lr] = dv.z; Ds[lc + 3][lr] = dv.w;
    Ts[lc + 0][lr] = tv.x; Ts[lc + 1][lr] = tv.y; Ts[lc + 2][lr] = tv.z; Ts[lc + 3][lr] = tv.w;
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      const float4 dp = *reinterpret_cast<const float4*>(&Ds[kk][ty * 4]);
      const float4 tp = *reinterpret_cast<const float4*>(&Ts[kk][tx * 4]);
      const float dd[4] = {dp.x, dp.y, dp.z, dp.w}, tt[4] = {tp.x, tp.y, tp.z, tp.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(dd[i], tt[j], acc[i][j]);
    }
    __syncthreads();
  }

  const int s = tile_struct[blockIdx.x];
  float flo[4] = {0, 0, 0, 0}, fhi[4] = {0, 0, 0, 0};
  float wlo[4], whi[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    wlo[j] = Weff[(long long)(k0 + tx * 4 + j) * 2 * S + 2 * s];
    whi[j] = Weff[(long long)(k0 + tx * 4 + j) * 2 * S + 2 * s + 1];
  }
  const float thr = DVH ? dvh_thr[s] : 0.f;
  float rv[4][4];
  int vcnt[4] = {0, 0, 0, 0};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int pr = p0 + ty * 4 + i;
    const float dl = pt_lo[pr], dh = pt_hi[pr];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float d = acc[i][j];
      rv[i][j] = 2.f * eq2_accumulate<float>(d, dl, dh, wlo[j], whi[j], flo[j], fhi[j]);
    }
    const int src = row_src[pr];
    if (dose_out && src >= 0) {
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (k0 + tx * 4 + j < K) dose_out[(long long)src * K + k0 + tx * 4 + j] = acc[i][j];
    }
    if (DVH && src >= 0) {
      const int sp = sel_pos[pr];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int k = k0 + tx * 4 + j;
        if (thr > 0.f && acc[i][j] >= thr) vcnt[j]++;
        if (sp >= 0) sel_buf[(long long)k * n_sel + sp] = acc[i][j];
      }
    }
  }
  if (DVH) {                       // integer counts: tile-level reduction, then one atomic per (tile, plan)
    __shared__ int redi[16][64];
#pragma unroll
    for (int j = 0; j < 4; ++j) redi[ty][tx * 4 + j] = vcnt[j];
    __syncthreads();
    if (tid < 64) {
      int sum = 0;
#pragma unroll
      for (int y = 0; y < 16; ++y) sum += redi[y][tid];
      if (sum) atomicAdd(&cnt[(long long)(k0 + tid) * S + s], sum);
    }
  }
  if (WRITE_R) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      float4 o = make_float4(rv[0][j], rv[1][j], rv[2][j], rv[3][j]);
      *reinterpret_cast<float4*>(R + (long long)(k0 + tx * 4 + j) * N_alloc + p0 + ty * 4) = o;
    }
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) { red[ty][tx * 4 + j][0] = flo[j]; red[ty][tx * 4 + j][1] = fhi[j]; }
  __syncthreads();
  if (tid < 128) {
    const int pl = tid >> 1, comp = tid & 1;
    float sum = 0.f;
#pragma unroll
    for (int y = 0; y < 16; ++y) sum += red[y][pl][comp];
    Fpart[((long long)blockIdx.x * K_pad + k0 + pl) * 2 + comp] = sum;
  }
}

int launch_simt_eval(const CaseDev& c, const PlanDev& p, bool write_R, float* dose_out, bool dvh_mode,
                     const float* dvh_thr, const int* gate, cudaStream_t st) {
  dim3 grid(c.N_alloc / 64, p.K_pad / 64);
  // rows beyond N_pad are all-zero padding with infinite thresholds: they contribute exactly 0
#define GMCO_SIMT_ARGS c.D, p.T, c.A_pad, c.N_alloc, p.K_pad, p.K, c.S, c.pt_lo, c.pt_hi, c.tile_struct, p.Weff, \
                       p.Fpart, p.R, dose_out, c.row_src, dvh_thr, p.res_cnt, c.sel_pos, p.res_sel, c.n_sel, gate
  if (dvh_mode)      k_simt_dose<false, true><<<grid, 256, 0, st>>>(GMCO_SIMT_ARGS);
  else if (write_R)  k_simt_dose<true, false><<<grid, 256, 0, st>>>(GMCO_SIMT_ARGS);
  else               k_simt_dose<false, false><<<grid, 256, 0, st>>>(GMCO_SIMT_ARGS);
#undef GMCO_SIMT_ARGS
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------
// a5 (SIMT): G[k][a] = sum_p R[k][p] D[p][a], 64 plans x 64 dwell per CTA, split over points.
__global__ void __launch_bounds__(256)
k_simt_grad(const float* __restrict__ R, const float* __restrict__ D, int A_pad, int N_alloc, int K_pad,
            int pts_per_split, float* __restrict__ Gpart, const int* __restrict__ gate) {
  if (gate && *gate == 0) return;
  __shared__ float Rs[16][68];
  __shared__ float Dsh[16][68];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int a0 = blockIdx.x * 64, k0 = blockIdx.y * 64;
  const int pb = blockIdx.z * pts_per_split, pe = min(pb + pts_per_split, N_alloc);
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  const int lr = tid >> 2, lc = (tid & 3) * 4;       // R loader: plan row 0..63, 4 consecutive points
  const int dr = tid >> 4, dc = (tid & 15) * 4;      // D loader: point row 0..15, 4 consecutive dwell
  for (int q0 = pb; q0 < pe; q0 += 16) {
    const float4 rv = *reinterpret_cast<const float4*>(R + (long long)(k0 + lr) * N_alloc + q0 + lc);
    Rs[lc + 0][lr] = rv.x; Rs[lc + 1][lr] = rv.y; Rs[lc + 2][lr] = rv.z; Rs[lc + 3][lr] = rv.w;
    float4 dv = make_float4(0.f, 0.f, 0.f, 0.f);
    if (a0 + dc < A_pad) dv = *reinterpret_cast<const float4*>(D + (long long)(q0 + dr) * A_pad + a0 + dc);
    *reinterpret_cast<float4*>(&Dsh[dr][dc]) = dv;
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      const float4 rp = *reinterpret_cast<const float4*>(&Rs[kk][ty * 4]);
      const float4 dp = *reinterpret_cast<const float4*>(&Dsh[kk][tx * 4]);
      const float rr[4] = {rp.x, rp.y, rp.z, rp.w}, dd[4] = {dp.x, dp.y, dp.z, dp.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(rr[i], dd[j], acc[i][j]);
    }
    __syncthreads();
  }
  if (a0 + tx * 4 < A_pad) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float4 o = make_float4(acc[i][0], acc[i][1], acc[i][2], acc[i][3]);
      *reinterpret_cast<float4*>(Gpart + ((long long)blockIdx.z * K_pad + k0 + ty * 4 + i) * A_pad + a0 + tx * 4) = o;
    }
  }
}

int launch_simt_grad(const CaseDev& c, const PlanDev& p, const int* gate, cudaStream_t st) {
  const int pts = ((c.N_alloc / 16 + p.nG - 1) / p.nG) * 16;
  dim3 grid((c.A_pad + 63) / 64, p.K_pad / 64, p.nG);
  k_simt_grad<<<grid, 256, 0, st>>>(p.R, c.D, c.A_pad, c.N_alloc, p.K_pad, pts, p.Gpart, gate);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------
// a8: per-plan D_level selection (nearest rank, descending) + V_level percentages + output packing.
// One CTA per plan.  Selection = 32-step bisection on the order-preserving integer image of fp32.
__device__ __forceinline__ uint32_t f2ord(float f) {
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t o) {
  return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}

struct ResultStructs {
  int n;
  int n_points[GMCO_MAX_STRUCTS], sel_begin[GMCO_MAX_STRUCTS], dvh_kind[GMCO_MAX_STRUCTS], rank[GMCO_MAX_STRUCTS];
  int tile_begin[GMCO_MAX_STRUCTS], tile_end[GMCO_MAX_STRUCTS];
};

__global__ void __launch_bounds__(256)
k_result(ResultStructs rs, float rx, int K, int K_pad, int A, int A_pad, int n_sel, const float* __restrict__ x,
         const float* __restrict__ Fpart /*[tile][K_pad][2]*/, const int* __restrict__ cnt,
         const float* __restrict__ sel, const int* __restrict__ it_done, const int* __restrict__ status,
         float* __restrict__ T_out, float* __restrict__ F_out, float* __restrict__ dvh_out,
         float* __restrict__ terms_out, int* __restrict__ iters_out, int* __restrict__ status_out) {
  const int k = blockIdx.x, tid = threadIdx.x;
  __shared__ int s_cnt;
  __shared__ float s_terms[2 * GMCO_MAX_STRUCTS];
  if (T_out)
    for (int a = tid; a < A; a += blockDim.x) { const float v = x[(long long)k * A_pad + a]; T_out[(long long)k * A + a] = v * v; }
  // objective terms: fixed-order sum over the tiles of each structure (deterministic)
  if (tid < 2 * rs.n) {
    const int s = tid >> 1, comp = tid & 1;
    float sum = 0.f;
    for (int t = rs.tile_begin[s]; t < rs.tile_end[s]; ++t) sum += Fpart[((long long)t * K_pad + k) * 2 + comp];
    s_terms[tid] = sum;
    if (terms_out) terms_out[(long long)k * 2 * rs.n + tid] = sum;
  }
  __syncthreads();
  if (tid == 0) {
    float F = 0.f;
    for (int i = 0; i < 2 * rs.n; ++i) F += s_terms[i];
    if (F_out) F_out[k] = F;
    if (iters_out) iters_out[k] = it_done[k];
    if (status_out) status_out[k] = status[k] == PLAN_RUNNING ? GMCO_PLAN_ITERS : status[k];
  }
  for (int s = 0; s < rs.n; ++s) {
    float val = 0.f;
    if (rs.dvh_kind[s] == 1) {
      val = 100.f * (float)cnt[(long long)k * rs.n + s] / (float)rs.n_points[s];
    } else if (rs.dvh_kind[s] == 2) {
      const float* v = sel + (long long)k * n_sel + rs.sel_begin[s];
      const int n = rs.n_points[s], rank = rs.rank[s];
      // largest ordinal o with count(v >= o) >= rank  ==  the rank-th largest value
      uint32_t o = 0;
      for (int bit = 31; bit >= 0; --bit) {
        const uint32_t cand = o | (1u << bit);
        if (tid == 0) s_cnt = 0;
        __syncthreads();
        int local = 0;
        for (int i = tid; i < n; i += blockDim.x) local += (f2ord(v[i]) >= cand);
        for (int off = 16; off; off >>= 1) local += __shfl_xor_sync(0xffffffffu, local, off);
        if ((tid & 31) == 0 && local) atomicAdd(&s_cnt, local);
        __syncthreads();
        if (s_cnt >= rank) o = cand;
        __syncthreads();
      }
      val = 100.f * ord2f(o) / rx;
    }
    if (tid == 0 && dvh_out) dvh_out[(long long)k * rs.n + s] = val;
  }
}

int launch_result(const CaseDev& c, const PlanDev& p, const StructHost* sh, float* T_out, float* F_out,
                  float* dvh_out, float* terms_out, int* iters_out, int* status_out, cudaStream_t st) {
  if (p.K == 0) return 0;
  ResultStructs rs{};
  rs.n = c.S;
  for (int s = 0; s < c.S; ++s) {
    rs.n_points[s] = sh[s].n_points; rs.sel_begin[s] = sh[s].sel_begin; rs.dvh_kind[s] = sh[s].dvh_kind;
    // nearest rank ceil(level/100 * n), reading A17 of DESIGN.md (double arithmetic, clamped to [1, n])
    long long r = (long long)ceil((double)sh[s].n_points * (double)sh[s].dvh_level / 100.0);
    if (r < 1) r = 1;
    if (r > sh[s].n_points) r = sh[s].n_points;
    rs.rank[s] = (int)r;
    rs.tile_begin[s] = sh[s].row_begin / 64; rs.tile_end[s] = (sh[s].row_begin + sh[s].n_rows_pad) / 64;
  }
  k_result<<<p.K, 256, 0, st>>>(rs, c.rx, p.K, p.K_pad, c.A, c.A_pad, c.n_sel, p.x, p.Fpart, p.res_cnt, p.res_sel,
                                p.it_done, p.status, T_out, F_out, dvh_out, terms_out, iters_out, status_out);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace gmco
