// S2 (chunk routing) and S3 (group refinement).
//
//   score_kernel : scores[b,kv,j,c] = <q_pooled[b,kv,j], chunk_sum[b,kv,c]> for the lower triangle c < j, as a tiled
//                  contraction with fp64 accumulation (inputs are fp32, converted once when staged in shared memory).
//                  Scores decide integer index sets that must match an fp64 oracle, so no TF32/bf16 tensor cores here.
//   select_fast_kernel (K_c <= 32) / select_generic_kernel: one warp per (b, kv, block j): top-K_c of the middle
//                  candidates by repeated warp arg-max
//                  (shuffle reduction on (score desc, index asc)), ascending compaction by ballot scan; then the
//                  C/g_s groups of every kept chunk are scored (warp-cooperative fp64 dot products) and the top-K_g kept.
#include <math_constants.h>

#include "hga_common.cuh"

namespace hga {

namespace {

constexpr int kTile = 64;
constexpr int kSlab = 32;

// 64 x 64 score tile per 64-thread CTA, 8 x 8 accumulators per thread: per k-step a thread reads 8 + 8 doubles for
// 64 DFMAs, which balances the shared-memory pipe against the fp64 pipe (a 4 x 4 micro-tile is LDS-bound 2:1).
// Thread (tx, ty) owns rows 16a + 2ty + {0,1} and columns 16b + 2tx + {0,1} (a, b = 0..3): every LDS.128 of a
// quarter-warp covers 128 contiguous bytes (S) or one broadcast address (Q).
__global__ void __launch_bounds__(64) score_kernel(const float* __restrict__ q_pooled, const float* __restrict__ chunk_sum,
                                                   float* __restrict__ scores, int n_b, int D, int F, int L_eff, int jb, int je) {
  // triangular tile index -> (tj, tc), tc <= tj
  const int ti = blockIdx.x;
  int tj = (int)((sqrtf(8.0f * (float)ti + 1.0f) - 1.0f) * 0.5f);
  while ((tj + 1) * (tj + 2) / 2 <= ti) ++tj;
  while (tj * (tj + 1) / 2 > ti) --tj;
  const int tc = ti - tj * (tj + 1) / 2;
  const int j0 = tj * kTile, c0 = tc * kTile;
  // any candidate (F <= c < j - L_eff) in this tile?  (block-uniform early exit)
  {
    const int jmax = min(j0 + kTile - 1, je - 1), cmin = max(c0, F);
    if (jmax < jb || j0 >= je) return;  // no row of [jb, je) in this tile (hga_prefill_window)
    if (cmin > jmax - L_eff - 1 || cmin > c0 + kTile - 1) return;
  }
  const size_t slice = (size_t)blockIdx.z * gridDim.y + blockIdx.y;  // b * Hkv + kv
  const float* Q = q_pooled + slice * (size_t)n_b * D;
  const float* S = chunk_sum + slice * (size_t)n_b * D;
  float* out = scores + slice * (size_t)n_b * n_b;

  __shared__ __align__(16) double Qs[kSlab][kTile];
  __shared__ __align__(16) double Ss[kSlab][kTile];
  const int tid = threadIdx.x, tx = tid % 8, ty = tid / 8;
  double acc[8][8];
#pragma unroll
  for (int a = 0; a < 8; ++a)
#pragma unroll
    for (int b = 0; b < 8; ++b) acc[a][b] = 0.0;

  for (int k0 = 0; k0 < D; k0 += kSlab) {
    __syncthreads();  // previous slab fully consumed
    {
      // thread `tid` stages row tid of both operands: 32 consecutive floats each, converted once to double
      const bool qok = j0 + tid < n_b, sok = c0 + tid < n_b;
      const float4* qp = reinterpret_cast<const float4*>(Q + (size_t)(j0 + tid) * D + k0);
      const float4* sp = reinterpret_cast<const float4*>(S + (size_t)(c0 + tid) * D + k0);
#pragma unroll
      for (int v4 = 0; v4 < kSlab / 4; ++v4) {
        const float4 qv = qok ? qp[v4] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 sv = sok ? sp[v4] : make_float4(0.f, 0.f, 0.f, 0.f);
        Qs[v4 * 4 + 0][tid] = (double)qv.x; Qs[v4 * 4 + 1][tid] = (double)qv.y;
        Qs[v4 * 4 + 2][tid] = (double)qv.z; Qs[v4 * 4 + 3][tid] = (double)qv.w;
        Ss[v4 * 4 + 0][tid] = (double)sv.x; Ss[v4 * 4 + 1][tid] = (double)sv.y;
        Ss[v4 * 4 + 2][tid] = (double)sv.z; Ss[v4 * 4 + 3][tid] = (double)sv.w;
      }
    }
    __syncthreads();
#pragma unroll 4
    for (int k = 0; k < kSlab; ++k) {
      double qa[8], sb[8];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const double2 qv = *reinterpret_cast<const double2*>(&Qs[k][16 * i + 2 * ty]);
        const double2 sv = *reinterpret_cast<const double2*>(&Ss[k][16 * i + 2 * tx]);
        qa[2 * i] = qv.x; qa[2 * i + 1] = qv.y;
        sb[2 * i] = sv.x; sb[2 * i + 1] = sv.y;
      }
#pragma unroll
      for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b] = fma(qa[a], sb[b], acc[a][b]);  // d ascending: fixed order
    }
  }
#pragma unroll
  for (int a = 0; a < 8; ++a) {
    const int j = j0 + 16 * (a / 2) + 2 * ty + (a % 2);
    if (j >= je || j < jb) continue;
#pragma unroll
    for (int b2 = 0; b2 < 4; ++b2) {
      const int c = c0 + 16 * b2 + 2 * tx;
      if (c + 1 < n_b && (n_b % 2) == 0) {
        *reinterpret_cast<float2*>(out + (size_t)j * n_b + c) = make_float2((float)acc[a][2 * b2], (float)acc[a][2 * b2 + 1]);
      } else {
        if (c < n_b) out[(size_t)j * n_b + c] = (float)acc[a][2 * b2];
        if (c + 1 < n_b) out[(size_t)j * n_b + c + 1] = (float)acc[a][2 * b2 + 1];
      }
    }
  }
}

// ----------------------------------------------------------------------------------------------------------------
// N3, R4's alternative (reading R19): score of a candidate = MAX over the block's 64*G rotated
// queries AS STORED of <q, S[cand]>, fp64 accumulation, d ascending.  One CTA = one (slice, block j, tile of 64
// candidates); it walks the G heads of the group, each a 64-row x 64-candidate x D contraction with the micro-tiling
// of score_kernel, and folds the rows away with a running max.  Candidates are either the dense chunk range
// [64 tc, 64 tc + 64) of chunk_sum (cand == nullptr) or rows of group_sum gathered through the kept chunks of the unit
// (group g = chunk_idx[a] * gpc + u for candidate a * gpc + u).  Exact but slow (fp64 SIMT over 64*G rows): the
// variant costs ~8 ms at c5 against 0.04 ms for the pooled-query rule.
// ----------------------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ float to_f32(T v);
template <>
__device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <>
__device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }

template <typename T>
__global__ void __launch_bounds__(64) score_max_kernel(const T* __restrict__ q_rot, const float* __restrict__ table,
                                                       const int32_t* __restrict__ chunk_idx, const int32_t* __restrict__ n_chunks,
                                                       float* __restrict__ out, int N, int n_b, int n_rows_tab, int D, int G, int Hkv,
                                                       int F, int L_eff, int jb, int Kc, int gpc, int out_stride, bool groups) {
  const int j = jb + (int)blockIdx.x;  // block of this CTA
  const int tc = blockIdx.y;                                          // candidate tile
  const size_t slice = blockIdx.z;                                    // b * Hkv + kv
  const size_t unit = slice * n_b + j;
  const int c0 = tc * kTile;
  int n_cand;  // candidates of this unit in candidate order
  if (groups) {
    n_cand = n_chunks[unit] * gpc;
  } else {
    n_cand = j - L_eff;  // dense chunk range [0, j - L_eff); entries below F are computed but never read
  }
  if (c0 >= n_cand) return;  // block-uniform
  __shared__ __align__(16) double Qs[kSlab][kTile];
  __shared__ __align__(16) double Ss[kSlab][kTile];
  __shared__ double red[8][kTile];
  const int tid = threadIdx.x, tx = tid % 8, ty = tid / 8;
  // row of `table` this thread stages (candidate c0 + tid)
  long long srow = -1;
  if (c0 + tid < n_cand) {
    if (groups) {
      const int cand = c0 + tid;
      srow = (long long)chunk_idx[unit * Kc + cand / gpc] * gpc + cand % gpc;
    } else {
      srow = c0 + tid;
    }
  }
  const float* S = table + slice * (size_t)n_rows_tab * D;
  const int b = (int)(slice / Hkv), kv = (int)(slice % Hkv);
  double best[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) best[i] = -CUDART_INF;
  for (int h = 0; h < G; ++h) {
    const T* Q = q_rot + (((size_t)b * Hkv * G + (size_t)kv * G + h) * N + (size_t)j * kChunk) * D;
    double acc[8][8];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
      for (int bb = 0; bb < 8; ++bb) acc[a][bb] = 0.0;
    for (int k0 = 0; k0 < D; k0 += kSlab) {
      __syncthreads();
      {
        const T* qp = Q + (size_t)tid * D + k0;
        const float* sp = S + (size_t)(srow < 0 ? 0 : srow) * D + k0;
#pragma unroll
        for (int u = 0; u < kSlab; ++u) {
          Qs[u][tid] = (double)to_f32<T>(qp[u]);
          Ss[u][tid] = srow < 0 ? 0.0 : (double)sp[u];
        }
      }
      __syncthreads();
#pragma unroll 4
      for (int k = 0; k < kSlab; ++k) {
        double qa[8], sb[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const double2 qv = *reinterpret_cast<const double2*>(&Qs[k][16 * i + 2 * ty]);
          const double2 sv = *reinterpret_cast<const double2*>(&Ss[k][16 * i + 2 * tx]);
          qa[2 * i] = qv.x; qa[2 * i + 1] = qv.y;
          sb[2 * i] = sv.x; sb[2 * i + 1] = sv.y;
        }
#pragma unroll
        for (int a = 0; a < 8; ++a)
#pragma unroll
          for (int bb = 0; bb < 8; ++bb) acc[a][bb] = fma(qa[a], sb[bb], acc[a][bb]);  // d ascending: fixed order
      }
    }
#pragma unroll
    for (int bb = 0; bb < 8; ++bb)
#pragma unroll
      for (int a = 0; a < 8; ++a) best[bb] = fmax(best[bb], acc[a][bb]);
  }
  // fold the 8 row-threads of every candidate column
#pragma unroll
  for (int b2 = 0; b2 < 4; ++b2) {
    red[ty][16 * b2 + 2 * tx] = best[2 * b2];
    red[ty][16 * b2 + 2 * tx + 1] = best[2 * b2 + 1];
  }
  __syncthreads();
  if (c0 + tid < n_cand) {
    double m = red[0][tid];
#pragma unroll
    for (int r = 1; r < 8; ++r) m = fmax(m, red[r][tid]);
    out[unit * (size_t)out_stride + c0 + tid] = (float)m;
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
__global__ void __launch_bounds__(128) select_generic_kernel(const float* __restrict__ scores, const float* __restrict__ q_pooled,
                                                     const float* __restrict__ group_sum, int32_t* __restrict__ chunk_idx,
                                                     float* __restrict__ chunk_score, int32_t* __restrict__ n_chunks,
                                                     int32_t* __restrict__ group_idx, float* __restrict__ group_score,
                                                     int32_t* __restrict__ n_groups, int n_units, int jb, int nj, int n_b, int n_g, int gpc,
                                                     int F, int L_eff, int Kc, int Kg, int kc_cap, int per_warp_floats,
                                                     int phase, const float* __restrict__ gscores_in) {
  // phase 0: chunk top-K_c, then group refinement with pooled-query scores; 1: chunks only; 2: groups only, from the
  // chunk lists already in chunk_idx / n_chunks and the candidate scores in gscores_in [unit][kc_cap * gpc] (N3 max rule)
  extern __shared__ __align__(16) float smem_f[];
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int widx = blockIdx.x * (blockDim.x / 32) + warp;
  if (widx >= n_units) return;  // warp-uniform; no block-wide barrier below
  float* work = smem_f + (size_t)warp * per_warp_floats;  // [n_b]
  float* gwork = work + n_b;                              // [kc_cap * gpc]
  float* gval = gwork + kc_cap * gpc;                     // [kc_cap * gpc]
  int* sel = reinterpret_cast<int*>(gval + kc_cap * gpc); // [kc_cap]

  const int j = jb + widx % nj;          // blocks [jb, jb + nj) of every slice
  const size_t slice = widx / nj;        // b * Hkv + kv
  const size_t unit = slice * n_b + j;   // row of every [B, Hkv, n_b, ...] table
  const float* row = scores + (size_t)unit * n_b;
  const int lo = F, hi = j - L_eff;
  const int n = hi > lo ? hi - lo : 0;
  int cnt = 0;
  int32_t* cidx = chunk_idx + (size_t)unit * Kc;
  float* csc = chunk_score ? chunk_score + (size_t)unit * Kc : nullptr;
  if (phase == 2) {
    cnt = n_chunks[unit];
    for (int c = lane; c < cnt; c += 32) sel[c] = cidx[c];
    __syncwarp();
  }
  if (phase != 2) for (int c = lane; c < n; c += 32) work[c] = row[lo + c];
  __syncwarp();
  const int take = min(Kc, n);
  if (phase != 2 && take < n) warp_topk_mark(work, n, take, lane);
  // ascending compaction of the marked candidates
  for (int c0 = 0; phase != 2 && c0 < n; c0 += 32) {
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
  if (phase != 2) {
    for (int s = cnt + lane; s < Kc; s += 32) {
      cidx[s] = -1;
      if (csc) csc[s] = 0.f;
    }
    if (n_chunks && lane == 0) n_chunks[unit] = cnt;
  }
  __syncwarp();
  if (Kg <= 0 || phase == 1) return;

  // group refinement: candidates in ascending group order (sel is ascending)
  const int n_gc = cnt * gpc;
  constexpr int VPL = D / 32;  // values per lane
  float qv[VPL];
  if (phase != 2) {
    const float* qp = q_pooled + (size_t)unit * D + lane * VPL;
#pragma unroll
    for (int u = 0; u < VPL; ++u) qv[u] = qp[u];
  } else {
#pragma unroll
    for (int u = 0; u < VPL; ++u) qv[u] = 0.f;
  }
  const float* gbase = group_sum + slice * (size_t)n_g * D;
  if (phase == 2) {
    for (int cand = lane; cand < n_gc; cand += 32) {
      const float v = gscores_in[unit * (size_t)(kc_cap * gpc) + cand];
      gwork[cand] = v;
      gval[cand] = v;
    }
  }
  for (int cand = 0; phase != 2 && cand < n_gc; ++cand) {
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

// ----------------------------------------------------------------------------------------------------------------
// Fast selection path (K_c <= 32, at most 128 group candidates): one warp per (b, kv, block j).
//   * the candidate row lives in shared memory with CONTIGUOUS ownership: lane l owns candidates [l*m, (l+1)*m)
//     (m a power of two, rows padded to m+4 floats so that the LDS.128 of a quarter-warp is conflict-free), and
//     keeps its best (value, offset) in registers;
//   * a round = one redux.sync max over order-preserving integer keys + a ballot (the lowest tied lane owns the
//     lowest index, R8) + a rescan of the winner lane's m candidates only;
//   * the <= 32 winners sit one per lane and are ranked ascending by index with 32 shuffles;
//   * group refinement scores one candidate per lane (fp64 FMA, d ascending, q in shared memory as doubles), so
//     there is no cross-lane reduction at all; its top-K_g uses the same redux rounds on <= 4 values per lane.
// ----------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t order_key(float v) {
  const uint32_t u = __float_as_uint(v + 0.0f);  // -0 -> +0, so equal floats have equal keys
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// Best (value, offset) of the m candidates at `col`; ascending scan with strict '>' keeps the lowest offset.
__device__ __forceinline__ void lane_rescan(const float* col, int m, float& bv, int& bo) {
  bv = -CUDART_INF_F;
  bo = 0;
  for (int o = 0; o < m; o += 4) {
    const float4 v = *reinterpret_cast<const float4*>(col + o);
    if (v.x > bv) { bv = v.x; bo = o; }
    if (v.y > bv) { bv = v.y; bo = o + 1; }
    if (v.z > bv) { bv = v.z; bo = o + 2; }
    if (v.w > bv) { bv = v.w; bo = o + 3; }
  }
}

template <int D>
__global__ void __launch_bounds__(128) select_fast_kernel(const float* __restrict__ scores, const float* __restrict__ q_pooled,
                                                          const float* __restrict__ group_sum, int32_t* __restrict__ chunk_idx,
                                                          float* __restrict__ chunk_score, int32_t* __restrict__ n_chunks,
                                                          int32_t* __restrict__ group_idx, float* __restrict__ group_score,
                                                          int32_t* __restrict__ n_groups, int n_units, int jb, int nj, int n_b, int n_g, int gpc,
                                                          int F, int L_eff, int Kc, int Kg, int lm, int per_warp_bytes) {
  extern __shared__ __align__(16) unsigned char smem_sel[];
  constexpr unsigned kFull = 0xffffffffu;
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int widx = blockIdx.x * (blockDim.x / 32) + warp;
  if (widx >= n_units) return;  // warp-uniform; no block-wide barrier below
  const int m = 1 << lm, stride = m + 4;
  unsigned char* base = smem_sel + (size_t)warp * per_warp_bytes;
  double* qd = reinterpret_cast<double*>(base);                 // [D]
  float* work = reinterpret_cast<float*>(base + D * 8);         // [32][m + 4]
  int* sel = reinterpret_cast<int*>(work + 32 * stride);        // [32]

  const int j = jb + widx % nj;          // blocks [jb, jb + nj) of every slice
  const size_t slice = widx / nj;        // b * Hkv + kv
  const size_t unit = slice * n_b + j;   // row of every [B, Hkv, n_b, ...] table
  const float* row = scores + (size_t)unit * n_b;
  const int lo = F, hi = j - L_eff;
  const int n = hi > lo ? hi - lo : 0;
  int32_t* cidx = chunk_idx + (size_t)unit * Kc;
  float* csc = chunk_score ? chunk_score + (size_t)unit * Kc : nullptr;

  // ---- stage the row (coalesced reads), pad with -inf -------------------------------------------------------
  const int n_lanes = (n + m - 1) >> lm;  // lanes that own at least one candidate
  for (int c = lane; c < n_lanes * m; c += 32) {
    const float v = c < n ? row[lo + c] : -CUDART_INF_F;
    work[(c >> lm) * stride + (c & (m - 1))] = v;
  }
  __syncwarp();
  float* col = work + lane * stride;
  float bv = -CUDART_INF_F;
  int bo = 0;
  if (lane < n_lanes) lane_rescan(col, m, bv, bo);

  // ---- top-K_c: one winner per round, kept in lane r ---------------------------------------------------------
  const int take = min(Kc, n);
  int win = 0x7fffffff;  // candidate index (relative to lo) of the winner this lane keeps
  float wsc = 0.f;
  if (take == n) {
    if (lane < n) {
      win = lane;
      wsc = work[(lane >> lm) * stride + (lane & (m - 1))];
    }
  } else {
    for (int r = 0; r < take; ++r) {
      const uint32_t key = order_key(bv);
      const uint32_t kmax = __reduce_max_sync(kFull, key);
      const int owner = __ffs(__ballot_sync(kFull, key == kmax)) - 1;
      const int cstar = __shfl_sync(kFull, lane * m + bo, owner);
      const float vstar = __shfl_sync(kFull, bv, owner);
      if (lane == r) {
        win = cstar;
        wsc = vstar;
      }
      if (lane == owner) {
        col[bo] = -CUDART_INF_F;
        lane_rescan(col, m, bv, bo);
      }
    }
  }
  // ---- ascending order: rank of this lane's winner among the winners ------------------------------------------
  int rank = 0;
#pragma unroll
  for (int t = 0; t < 32; ++t) rank += (__shfl_sync(kFull, win, t) < win) ? 1 : 0;
  const int cnt = take;
  if (lane < cnt) {
    cidx[rank] = lo + win;
    sel[rank] = lo + win;
    if (csc) csc[rank] = wsc;
  }
  for (int s = cnt + lane; s < Kc; s += 32) {
    cidx[s] = -1;
    if (csc) csc[s] = 0.f;
  }
  if (n_chunks && lane == 0) n_chunks[unit] = cnt;
  if (Kg <= 0) return;

  // ---- group refinement: candidate `cand` = group cand % gpc of kept chunk cand / gpc (ascending group order) -----
  const int n_gc = cnt * gpc;  // <= 128
  {
    const float* qp = q_pooled + (size_t)unit * D;
    for (int d = lane; d < D; d += 32) qd[d] = (double)qp[d];
  }
  __syncwarp();
  const float* gbase = group_sum + slice * (size_t)n_g * D;
  float gsc[4];   // score of candidate lane + 32*i
  int gid[4];     // its group index
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int cand = lane + 32 * i;
    gsc[i] = -CUDART_INF_F;
    gid[i] = -1;
    if (cand < n_gc) {
      const int g = sel[cand / gpc] * gpc + cand % gpc;
      const float4* gp = reinterpret_cast<const float4*>(gbase + (size_t)g * D);
      double s = 0.0;
#pragma unroll 4
      for (int d4 = 0; d4 < D / 4; ++d4) {
        const float4 v = __ldg(gp + d4);
        const double2 q01 = *reinterpret_cast<const double2*>(qd + 4 * d4);
        const double2 q23 = *reinterpret_cast<const double2*>(qd + 4 * d4 + 2);
        s = fma(q01.x, (double)v.x, s);
        s = fma(q01.y, (double)v.y, s);
        s = fma(q23.x, (double)v.z, s);
        s = fma(q23.y, (double)v.w, s);
      }
      gsc[i] = (float)s;
      gid[i] = g;
    }
  }
  const int gtake = min(Kg, n_gc);
  unsigned taken = 0;  // bit i: candidate lane + 32*i is kept
  if (gtake == n_gc) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
      if (lane + 32 * i < n_gc) taken |= 1u << i;
  } else {
    float wv[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) wv[i] = gsc[i];
    for (int r = 0; r < gtake; ++r) {
      // lane-local best: value descending, candidate index ascending (i ascending == index ascending)
      float lv = wv[0];
      int li = 0;
#pragma unroll
      for (int i = 1; i < 4; ++i)
        if (wv[i] > lv) { lv = wv[i]; li = i; }
      const uint32_t key = order_key(lv);
      const uint32_t kmax = __reduce_max_sync(kFull, key);
      const bool tied = key == kmax;
      const uint32_t cmin = __reduce_min_sync(kFull, tied ? (uint32_t)(lane + 32 * li) : 0xffffffffu);
      if (tied && (uint32_t)(lane + 32 * li) == cmin) {
        taken |= 1u << li;
#pragma unroll
        for (int i = 0; i < 4; ++i)
          if (i == li) wv[i] = -CUDART_INF_F;
      }
    }
  }
  // ascending compaction (candidates are in ascending group order)
  int gcnt = 0;
  int32_t* gidx = group_idx + (size_t)unit * Kg;
  float* gscore = group_score ? group_score + (size_t)unit * Kg : nullptr;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const bool on = (taken >> i) & 1u;
    const unsigned mk = __ballot_sync(kFull, on);
    if (on) {
      const int pos = gcnt + __popc(mk & ((1u << lane) - 1u));
      gidx[pos] = gid[i];
      if (gscore) gscore[pos] = gsc[i];
    }
    gcnt += __popc(mk);
  }
  for (int s = gcnt + lane; s < Kg; s += 32) {
    gidx[s] = -1;
    if (gscore) gscore[s] = 0.f;
  }
  if (n_groups && lane == 0) n_groups[unit] = gcnt;
}

}  // namespace

hga_status launch_route(const Derived& d, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                        int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                        float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s) {
  const int nt = (d.n_b + kTile - 1) / kTile;
  dim3 grid(nt * (nt + 1) / 2, d.Hkv, d.B);
  score_kernel<<<grid, 64, 0, s>>>(q_pooled, chunk_sum, score_ws, d.n_b, d.D, d.F, d.L_eff, d.jb, d.jb + d.nj);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;

  const int n_units = d.B * d.Hkv * d.nj;
  const int kc_cap = d.Kc < d.n_b ? (d.Kc > 0 ? d.Kc : 1) : d.n_b;
  if (d.Kc <= 32 && kc_cap * d.gpc <= 128) {
    // fast path: register/redux rounds, one candidate per lane in the group stage
    const int n_max = d.n_b - d.F - d.L_eff > 1 ? d.n_b - d.F - d.L_eff : 1;
    int lm = 2;
    while ((32 << lm) < n_max) ++lm;
    const int per_warp_bytes = d.D * 8 + 32 * ((1 << lm) + 4) * 4 + 32 * 4;
    int warps = 4;
    while (warps > 1 && (size_t)warps * per_warp_bytes > 200 * 1024) warps >>= 1;
    const size_t smem = (size_t)warps * per_warp_bytes;
    if (smem <= 200 * 1024) {
      auto kern = d.D == 128 ? select_fast_kernel<128> : select_fast_kernel<64>;
      HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      kern<<<(n_units + warps - 1) / warps, warps * 32, smem, s>>>(score_ws, q_pooled, group_sum, chunk_idx, chunk_score,
                                                                   n_chunks, group_idx, group_score, n_groups, n_units,
                                                                   d.jb, d.nj, d.n_b, d.n_g, d.gpc, d.F, d.L_eff, d.Kc, d.Kg, lm,
                                                                   per_warp_bytes);
      return launch_status();
    }
  }
  const int per_warp = d.n_b + 2 * kc_cap * d.gpc + kc_cap;
  int warps = 4;
  while (warps > 1 && (size_t)warps * per_warp * sizeof(float) > 200 * 1024) warps >>= 1;
  const size_t smem = (size_t)warps * per_warp * sizeof(float);
  if (smem > 200 * 1024) return HGA_ERR_UNSUPPORTED;
  auto kern = d.D == 128 ? select_generic_kernel<128> : select_generic_kernel<64>;
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<(n_units + warps - 1) / warps, warps * 32, smem, s>>>(score_ws, q_pooled, group_sum, chunk_idx, chunk_score,
                                                               n_chunks, group_idx, group_score, n_groups, n_units, d.jb, d.nj, d.n_b,
                                                               d.n_g, d.gpc, d.F, d.L_eff, d.Kc, d.Kg, kc_cap, per_warp, 0, nullptr);
  return launch_status();
}

// N3 max rule: chunk scores (max over the block's stored rotated queries) -> top-K_c -> group candidate scores of the
// kept chunks -> top-K_g.  score_ws: [B, Hkv, n_b, n_b] chunk scores followed by [B, Hkv, n_b, kc_cap * gpc] group scores.
hga_status launch_route_max(const Derived& d, const void* q_rot, const float* chunk_sum, const float* group_sum,
                            int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                            float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s) {
  const int n_units = d.B * d.Hkv * d.nj;
  const int kc_cap = d.Kc < d.n_b ? (d.Kc > 0 ? d.Kc : 1) : d.n_b;
  float* gscores = score_ws + (size_t)d.B * d.Hkv * d.n_b * d.n_b;
  const int per_warp = d.n_b + 2 * kc_cap * d.gpc + kc_cap;
  int warps = 4;
  while (warps > 1 && (size_t)warps * per_warp * sizeof(float) > 200 * 1024) warps >>= 1;
  const size_t smem = (size_t)warps * per_warp * sizeof(float);
  if (smem > 200 * 1024) return HGA_ERR_UNSUPPORTED;
  auto sel = d.D == 128 ? select_generic_kernel<128> : select_generic_kernel<64>;
  HGA_CUDA_OK(cudaFuncSetAttribute(sel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int ct = (d.n_b + kTile - 1) / kTile, gt = (kc_cap * d.gpc + kTile - 1) / kTile;
  auto run_scores = [&](bool groups, const float* table, int n_rows_tab, float* out, int out_stride, int tiles) {
    dim3 grid(d.nj, tiles, d.B * d.Hkv);
    if (d.bf16_io)
      score_max_kernel<__nv_bfloat16><<<grid, 64, 0, s>>>((const __nv_bfloat16*)q_rot, table, chunk_idx, n_chunks, out, d.N, d.n_b,
                                                          n_rows_tab, d.D, d.G, d.Hkv, d.F, d.L_eff, d.jb, d.Kc, d.gpc, out_stride, groups);
    else
      score_max_kernel<float><<<grid, 64, 0, s>>>((const float*)q_rot, table, chunk_idx, n_chunks, out, d.N, d.n_b, n_rows_tab,
                                                  d.D, d.G, d.Hkv, d.F, d.L_eff, d.jb, d.Kc, d.gpc, out_stride, groups);
  };
  run_scores(false, chunk_sum, d.n_b, score_ws, d.n_b, ct);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
  sel<<<(n_units + warps - 1) / warps, warps * 32, smem, s>>>(score_ws, nullptr, group_sum, chunk_idx, chunk_score, n_chunks,
                                                              group_idx, group_score, n_groups, n_units, d.jb, d.nj, d.n_b, d.n_g,
                                                              d.gpc, d.F, d.L_eff, d.Kc, d.Kg, kc_cap, per_warp, 1, nullptr);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
  if (d.Kg <= 0) return HGA_OK;
  run_scores(true, group_sum, d.n_g, gscores, kc_cap * d.gpc, gt);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
  sel<<<(n_units + warps - 1) / warps, warps * 32, smem, s>>>(score_ws, nullptr, group_sum, chunk_idx, chunk_score, n_chunks,
                                                              group_idx, group_score, n_groups, n_units, d.jb, d.nj, d.n_b, d.n_g,
                                                              d.gpc, d.F, d.L_eff, d.Kc, d.Kg, kc_cap, per_warp, 2, gscores);
  return launch_status();
}

}  // namespace hga
