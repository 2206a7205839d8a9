// S2 (chunk routing) and S3 (group refinement).
//
//   score_kernel : scores[b,kv,j,c] = <q_pooled[b,kv,j], chunk_sum[b,kv,c]> for the lower triangle c < j, as a tiled
//                  contraction with fp64 accumulation (inputs are fp32, converted once when staged in shared memory).
//                  Scores decide integer index sets that must match an fp64 oracle, so no TF32/bf16 tensor cores here.
//   select_kernel: one warp per (b, kv, block j): top-K_c of the middle candidates by repeated warp arg-max
//                  (shuffle reduction on (score desc, index asc)), ascending compaction by ballot scan; then the
//                  C/g_s groups of every kept chunk are scored (warp-cooperative fp64 dot products) and the top-K_g kept.
#include <math_constants.h>

#include "hga_common.cuh"

namespace hga {

namespace {

constexpr int kTile = 64;
constexpr int kSlab = 16;

__global__ void __launch_bounds__(256) score_kernel(const float* __restrict__ q_pooled, const float* __restrict__ chunk_sum,
                                                    float* __restrict__ scores, int n_b, int D, int F, int L_eff) {
  // triangular tile index -> (tj, tc), tc <= tj
  const int ti = blockIdx.x;
  int tj = (int)((sqrtf(8.0f * (float)ti + 1.0f) - 1.0f) * 0.5f);
  while ((tj + 1) * (tj + 2) / 2 <= ti) ++tj;
  while (tj * (tj + 1) / 2 > ti) --tj;
  const int tc = ti - tj * (tj + 1) / 2;
  const int j0 = tj * kTile, c0 = tc * kTile;
  // any candidate (F <= c < j - L_eff) in this tile?  (block-uniform early exit)
  {
    const int jmax = min(j0 + kTile - 1, n_b - 1), cmin = max(c0, F);
    if (cmin > jmax - L_eff - 1 || cmin > c0 + kTile - 1) return;
  }
  const size_t slice = (size_t)blockIdx.z * gridDim.y + blockIdx.y;  // b * Hkv + kv
  const float* Q = q_pooled + slice * (size_t)n_b * D;
  const float* S = chunk_sum + slice * (size_t)n_b * D;
  float* out = scores + slice * (size_t)n_b * n_b;

  __shared__ __align__(16) double Qs[kSlab][kTile + 2];
  __shared__ __align__(16) double Ss[kSlab][kTile + 2];
  const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
  const int lr = threadIdx.x / 4, lp = threadIdx.x % 4;  // loader: row, float4 part of the 16-wide slab
  double acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;

  for (int k0 = 0; k0 < D; k0 += kSlab) {
    float4 qv = make_float4(0.f, 0.f, 0.f, 0.f), sv = qv;
    if (j0 + lr < n_b) qv = *reinterpret_cast<const float4*>(Q + (size_t)(j0 + lr) * D + k0 + lp * 4);
    if (c0 + lr < n_b) sv = *reinterpret_cast<const float4*>(S + (size_t)(c0 + lr) * D + k0 + lp * 4);
    __syncthreads();  // previous slab fully consumed
    Qs[lp * 4 + 0][lr] = (double)qv.x; Qs[lp * 4 + 1][lr] = (double)qv.y;
    Qs[lp * 4 + 2][lr] = (double)qv.z; Qs[lp * 4 + 3][lr] = (double)qv.w;
    Ss[lp * 4 + 0][lr] = (double)sv.x; Ss[lp * 4 + 1][lr] = (double)sv.y;
    Ss[lp * 4 + 2][lr] = (double)sv.z; Ss[lp * 4 + 3][lr] = (double)sv.w;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kSlab; ++k) {
      double2 q01 = *reinterpret_cast<const double2*>(&Qs[k][ty * 4]);
      double2 q23 = *reinterpret_cast<const double2*>(&Qs[k][ty * 4 + 2]);
      double2 s01 = *reinterpret_cast<const double2*>(&Ss[k][tx * 4]);
      double2 s23 = *reinterpret_cast<const double2*>(&Ss[k][tx * 4 + 2]);
      const double qa[4] = {q01.x, q01.y, q23.x, q23.y};
      const double sb[4] = {s01.x, s01.y, s23.x, s23.y};
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = fma(qa[a], sb[b], acc[a][b]);  // d ascending: fixed order
    }
  }
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const int j = j0 + ty * 4 + a;
    const int c = c0 + tx * 4;
    if (j < n_b && c < n_b)  // n_b % 4 may be nonzero only for tiny problems; guard element-wise then
    {
      if (c + 3 < n_b && (n_b % 4) == 0) {
        *reinterpret_cast<float4*>(out + (size_t)j * n_b + c) =
            make_float4((float)acc[a][0], (float)acc[a][1], (float)acc[a][2], (float)acc[a][3]);
      } else {
        for (int b = 0; b < 4 && c + b < n_b; ++b) out[(size_t)j * n_b + c + b] = (float)acc[a][b];
      }
    }
  }
}

// Mark the `take` best of work[0..n) by overwriting them with -inf.  Order: score descending, index ascending (R8).
__device__ __forceinline__ void warp_topk_mark(float* work, int n, int take, int lane) {
  for (int r = 0; r < take; ++r) {
    float bv = -CUDART_INF_F;
    int bi = 0x7fffffff;
    for (int c = lane; c < n; c += 32) {
      float v = work[c];
      if (v > bv) { bv = v; bi = c; }  // ascending scan + strict '>' keeps the lowest index among equals
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      float ov = __shfl_xor_sync(0xffffffffu, bv, off);
      int oi = __shfl_xor_sync(0xffffffffu, bi, off);
      if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if ((bi & 31) == lane && bi < n) work[bi] = -CUDART_INF_F;
    __syncwarp();
  }
}

template <int D>
__global__ void __launch_bounds__(128) select_kernel(const float* __restrict__ scores, const float* __restrict__ q_pooled,
                                                     const float* __restrict__ group_sum, int32_t* __restrict__ chunk_idx,
                                                     float* __restrict__ chunk_score, int32_t* __restrict__ n_chunks,
                                                     int32_t* __restrict__ group_idx, float* __restrict__ group_score,
                                                     int32_t* __restrict__ n_groups, int n_units, int n_b, int n_g, int gpc,
                                                     int F, int L_eff, int Kc, int Kg, int kc_cap, int per_warp_floats) {
  extern __shared__ __align__(16) float smem_f[];
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int unit = blockIdx.x * (blockDim.x / 32) + warp;
  if (unit >= n_units) return;  // warp-uniform; no block-wide barrier below
  float* work = smem_f + (size_t)warp * per_warp_floats;  // [n_b]
  float* gwork = work + n_b;                              // [kc_cap * gpc]
  float* gval = gwork + kc_cap * gpc;                     // [kc_cap * gpc]
  int* sel = reinterpret_cast<int*>(gval + kc_cap * gpc); // [kc_cap]

  const int j = unit % n_b;
  const size_t slice = unit / n_b;  // b * Hkv + kv
  const float* row = scores + (size_t)unit * n_b;
  const int lo = F, hi = j - L_eff;
  const int n = hi > lo ? hi - lo : 0;
  for (int c = lane; c < n; c += 32) work[c] = row[lo + c];
  __syncwarp();
  const int take = min(Kc, n);
  if (take < n) warp_topk_mark(work, n, take, lane);
  // ascending compaction of the marked candidates
  int cnt = 0;
  int32_t* cidx = chunk_idx + (size_t)unit * Kc;
  float* csc = chunk_score ? chunk_score + (size_t)unit * Kc : nullptr;
  for (int c0 = 0; c0 < n; c0 += 32) {
    const int c = c0 + lane;
    const bool on = c < n && (take == n || work[c] == -CUDART_INF_F);
    const unsigned m = __ballot_sync(0xffffffffu, on);
    if (on) {
      const int pos = cnt + __popc(m & ((1u << lane) - 1u));
      cidx[pos] = lo + c;
      sel[pos] = lo + c;
      if (csc) csc[pos] = row[lo + c];
    }
    cnt += __popc(m);
  }
  for (int s = cnt + lane; s < Kc; s += 32) {
    cidx[s] = -1;
    if (csc) csc[s] = 0.f;
  }
  if (n_chunks && lane == 0) n_chunks[unit] = cnt;
  __syncwarp();
  if (Kg <= 0) return;

  // group refinement: candidates in ascending group order (sel is ascending)
  const int n_gc = cnt * gpc;
  constexpr int VPL = D / 32;  // values per lane
  float qv[VPL];
  {
    const float* qp = q_pooled + (size_t)unit * D + lane * VPL;
#pragma unroll
    for (int u = 0; u < VPL; ++u) qv[u] = qp[u];
  }
  const float* gbase = group_sum + slice * (size_t)n_g * D;
  for (int cand = 0; cand < n_gc; ++cand) {
    const int g = sel[cand / gpc] * gpc + cand % gpc;
    const float* gp = gbase + (size_t)g * D + lane * VPL;
    double s = 0.0;
#pragma unroll
    for (int u = 0; u < VPL; ++u) s = fma((double)qv[u], (double)gp[u], s);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if (lane == 0) {
      gwork[cand] = (float)s;
      gval[cand] = (float)s;
    }
  }
  __syncwarp();
  const int gtake = min(Kg, n_gc);
  if (gtake < n_gc) warp_topk_mark(gwork, n_gc, gtake, lane);
  int gcnt = 0;
  int32_t* gidx = group_idx + (size_t)unit * Kg;
  float* gsc = group_score ? group_score + (size_t)unit * Kg : nullptr;
  for (int c0 = 0; c0 < n_gc; c0 += 32) {
    const int c = c0 + lane;
    const bool on = c < n_gc && (gtake == n_gc || gwork[c] == -CUDART_INF_F);
    const unsigned m = __ballot_sync(0xffffffffu, on);
    if (on) {
      const int pos = gcnt + __popc(m & ((1u << lane) - 1u));
      gidx[pos] = sel[c / gpc] * gpc + c % gpc;
      if (gsc) gsc[pos] = gval[c];
    }
    gcnt += __popc(m);
  }
  for (int s = gcnt + lane; s < Kg; s += 32) {
    gidx[s] = -1;
    if (gsc) gsc[s] = 0.f;
  }
  if (n_groups && lane == 0) n_groups[unit] = gcnt;
}

}  // namespace

hga_status launch_route(const Derived& d, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                        int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                        float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s) {
  const int nt = (d.n_b + kTile - 1) / kTile;
  dim3 grid(nt * (nt + 1) / 2, d.Hkv, d.B);
  score_kernel<<<grid, 256, 0, s>>>(q_pooled, chunk_sum, score_ws, d.n_b, d.D, d.F, d.L_eff);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;

  const int n_units = d.B * d.Hkv * d.n_b;
  const int kc_cap = d.Kc < d.n_b ? (d.Kc > 0 ? d.Kc : 1) : d.n_b;
  const int per_warp = d.n_b + 2 * kc_cap * d.gpc + kc_cap;
  int warps = 4;
  while (warps > 1 && (size_t)warps * per_warp * sizeof(float) > 200 * 1024) warps >>= 1;
  const size_t smem = (size_t)warps * per_warp * sizeof(float);
  if (smem > 200 * 1024) return HGA_ERR_UNSUPPORTED;
  auto kern = d.D == 128 ? select_kernel<128> : select_kernel<64>;
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<(n_units + warps - 1) / warps, warps * 32, smem, s>>>(score_ws, q_pooled, group_sum, chunk_idx, chunk_score,
                                                               n_chunks, group_idx, group_score, n_groups, n_units, d.n_b,
                                                               d.n_g, d.gpc, d.F, d.L_eff, d.Kc, d.Kg, kc_cap, per_warp);
  return launch_status();
}

}  // namespace hga
