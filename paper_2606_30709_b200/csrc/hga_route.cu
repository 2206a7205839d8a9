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

#include <mutex>
#include <type_traits>

#include "hga_common.cuh"
#include "hga_tc_ptx.cuh"

namespace hga {

namespace {

// -DHGA_ROUTE_TRACE: cycles per phase summed over the CTAs of score_max_listed_kernel (slots 0-7, count in 15) and over the
// warps of select_fast_kernel (slots 16-23, count in 31); read back by hga_debug_route_trace
#ifdef HGA_ROUTE_TRACE
__device__ unsigned long long g_rt[32];
#define HGA_RT_BEGIN long long t0_ = clock64()
#define HGA_RT(i)                                                        \
  do {                                                                   \
    if (threadIdx.x % 32 == 0 && ((i) >= 16 || threadIdx.x == 0)) {      \
      const long long t_ = clock64();                                    \
      atomicAdd(&g_rt[i], (unsigned long long)(t_ - t0_));               \
      t0_ = t_;                                                          \
    }                                                                    \
  } while (0)
#else
#define HGA_RT_BEGIN do { } while (0)
#define HGA_RT(i) do { } while (0)
#endif

constexpr int kTile = 64;
constexpr int kSlab = 32;

// 64 x 64 score tile per 128-thread CTA on the fp64 tensor-core instruction (mma.sync.m8n8k4.f64): warp (wr, wc) owns the
// 32 x 32 quadrant, i.e. 4 x 4 fragments of 8 x 8, 32 accumulator doubles per thread.  DMMA runs at the DFMA rate (64 FMA per
// clock and SM, csrc/microbench/fp64_throughput.cu) but takes its operands once per warp: a k = 4 step costs a thread 8 doubles
// from shared memory for 128 FMAs, where the DFMA micro-tiles cost 12 (4 x 8 tile) or 16 (8 x 8) doubles for 32 / 64 -- and
// the register-file return path of shared memory (128 B per clock and SM) was what bound those forms (ncu: 5.6 M wavefronts
// against 4.5 M cycles of fp64 work, fp64 pipe 45 % active).  Products and sums are fp64 as before; the order of the four
// products inside one instruction is the hardware's (the result is compared with the oracle at 1e-6 relative, R15).
// Shared layout [k][row] with a row pitch of 72 doubles: the four k-rows of a fragment fall into two disjoint bank halves.
constexpr int kPitch = kTile + 8;

__device__ __forceinline__ void dmma_8x8x4(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(128) score_kernel(const float* __restrict__ q_pooled, const float* __restrict__ chunk_sum,
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
  // the workspace holds the rows of [jb, je) only: row (slice, j) at (slice * (je - jb) + j - jb) * n_b
  float* out = scores + (slice * (size_t)(je - jb) - (size_t)jb) * n_b;

  __shared__ __align__(16) double Qs[kSlab][kPitch];
  __shared__ __align__(16) double Ss[kSlab][kPitch];
  const int tid = threadIdx.x, lane = tid % 32, warp = tid / 32;
  const int wr = (warp / 2) * 32, wc = (warp % 2) * 32;  // this warp's quadrant of the tile
  const int fr = lane / 4, fk = lane % 4;                // fragment coordinates of this lane
  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // threads 0..63 stage row tid of Q, threads 64..127 row tid - 64 of S: 32 consecutive floats per slab, converted once; the
  // next slab's floats are fetched into registers before the current slab is consumed
  const int rr = tid & 63;
  const bool is_q = tid < 64;
  const int srow = (is_q ? j0 : c0) + rr;
  const bool ok = srow < n_b;
  const float4* src = reinterpret_cast<const float4*>((is_q ? Q : S) + (size_t)srow * D);
  double(*dst)[kPitch] = is_q ? Qs : Ss;
  float4 pre[kSlab / 4];
#pragma unroll
  for (int v4 = 0; v4 < kSlab / 4; ++v4) pre[v4] = ok ? src[v4] : make_float4(0.f, 0.f, 0.f, 0.f);
  for (int k0 = 0; k0 < D; k0 += kSlab) {
    __syncthreads();  // previous slab fully consumed
#pragma unroll
    for (int v4 = 0; v4 < kSlab / 4; ++v4) {
      dst[v4 * 4 + 0][rr] = (double)pre[v4].x; dst[v4 * 4 + 1][rr] = (double)pre[v4].y;
      dst[v4 * 4 + 2][rr] = (double)pre[v4].z; dst[v4 * 4 + 3][rr] = (double)pre[v4].w;
    }
    if (k0 + kSlab < D) {
#pragma unroll
      for (int v4 = 0; v4 < kSlab / 4; ++v4) pre[v4] = ok ? src[(k0 + kSlab) / 4 + v4] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();
#pragma unroll 2
    for (int k = 0; k < kSlab; k += 4) {  // d ascending in steps of four
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        a[i] = Qs[k + fk][wr + 8 * i + fr];  // A[row][k]: row = lane / 4, k = lane % 4
        b[i] = Ss[k + fk][wc + 8 * i + fr];  // B[k][col]: k = lane % 4, col = lane / 4
      }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma_8x8x4(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
  }
  // C fragment: row = lane / 4, columns 2 (lane % 4) + {0, 1}
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int j = j0 + wr + 8 * i + fr;
    if (j >= je || j < jb) continue;
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {
      const int c = c0 + wc + 8 * jj + 2 * fk;
      if (c + 1 < n_b && (n_b % 2) == 0) {
        *reinterpret_cast<float2*>(out + (size_t)j * n_b + c) = make_float2((float)acc[i][jj][0], (float)acc[i][jj][1]);
      } else {
        if (c < n_b) out[(size_t)j * n_b + c] = (float)acc[i][jj][0];
        if (c + 1 < n_b) out[(size_t)j * n_b + c + 1] = (float)acc[i][jj][1];
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
                                                       int F, int L_eff, int jb, int Kc, int gpc, int out_stride, bool groups,
                                                       const int32_t* __restrict__ only_neg) {
  const int j = jb + (int)blockIdx.x;  // block of this CTA
  const int tc = blockIdx.y;                                          // candidate tile
  const size_t slice = blockIdx.z;                                    // b * Hkv + kv
  const size_t unit = slice * n_b + j;
  if (only_neg != nullptr && only_neg[unit] >= 0) return;  // block-uniform: only the flagged units are recomputed
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
                                                     int phase, const float* __restrict__ gscores_in,
                                                     const int32_t* __restrict__ only_neg) {
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
  if (only_neg != nullptr && only_neg[unit] >= 0) return;  // warp-uniform
  // mean rule (phase 0): the workspace holds the rows of [jb, jb + nj) only; max rule: the full [B, Hkv, n_b, n_b] matrix
  const float* row = scores + (size_t)(phase == 0 ? (size_t)widx : unit) * n_b;
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

// Best (value, offset) of the m candidates at `col` (m a multiple of 4): the maximum by a max tree, then the lowest
// offset that holds it (descending scan of independent equality tests: the last write is the lowest offset, R8).
__device__ __forceinline__ void lane_rescan(const float* col, int m, float& bv, int& bo) {
  if (m <= 8) {  // short runs: one ascending pass with strict '>' (keeps the lowest offset) beats two passes
    bv = -CUDART_INF_F;
    bo = 0;
    for (int o = 0; o < m; o += 4) {
      const float4 v = *reinterpret_cast<const float4*>(col + o);
      if (v.x > bv) { bv = v.x; bo = o; }
      if (v.y > bv) { bv = v.y; bo = o + 1; }
      if (v.z > bv) { bv = v.z; bo = o + 2; }
      if (v.w > bv) { bv = v.w; bo = o + 3; }
    }
    return;
  }
  float b0 = -CUDART_INF_F, b1 = -CUDART_INF_F;
  for (int o = 0; o < m; o += 4) {
    const float4 v = *reinterpret_cast<const float4*>(col + o);
    b0 = tc::max3(b0, v.x, v.y);
    b1 = tc::max3(b1, v.z, v.w);
  }
  bv = fmaxf(b0, b1);
  bo = 0;
  for (int o = m - 4; o >= 0; o -= 4) {
    const float4 v = *reinterpret_cast<const float4*>(col + o);
    if (v.w == bv) bo = o + 3;
    if (v.z == bv) bo = o + 2;
    if (v.y == bv) bo = o + 1;
    if (v.x == bv) bo = o;
  }
}

// Register-resident form of lane_rescan for a lane that keeps its M candidates in registers (static indexing only).
template <int M>
__device__ __forceinline__ void reg_rescan(const float (&v)[M], float& bv, int& bo) {
  float b0 = -CUDART_INF_F, b1 = -CUDART_INF_F;
#pragma unroll
  for (int o = 0; o < M; o += 4) {
    b0 = tc::max3(b0, v[o], v[o + 1]);
    b1 = tc::max3(b1, v[o + 2], v[o + 3]);
  }
  bv = fmaxf(b0, b1);
  bo = 0;
#pragma unroll
  for (int o = M - 1; o >= 0; --o)
    if (v[o] == bv) bo = o;  // the last write is the lowest offset (R8)
}

// M > 0: every lane keeps its run of M = 2^lm candidates in registers during the top-K_c rounds (the owner of a round's
// winner removes it and rescans without touching shared memory: c5 route 73 -> 69 us, c4 46 -> 44 us); M == 0: the run
// lives in shared memory (any lm; runs of 8 and shorter measured no gain in registers).
template <int D, int M>
__global__ void __launch_bounds__(128, (M > 0 ? 7 : 9)) select_fast_kernel(const float* __restrict__ scores, const float* __restrict__ q_pooled,
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
  float* work = reinterpret_cast<float*>(base);                 // [32][m + 4]; after the chunk stage: the query as doubles [D]
  int* sel = reinterpret_cast<int*>(work + 32 * stride);        // [32]

  const int j = jb + widx % nj;          // blocks [jb, jb + nj) of every slice
  const size_t slice = widx / nj;        // b * Hkv + kv
  const size_t unit = slice * n_b + j;   // row of every [B, Hkv, n_b, ...] table
  const float* row = scores + (size_t)widx * n_b;  // the score workspace holds the rows of [jb, jb + nj) only
  const int lo = F, hi = j - L_eff;
  const int n = hi > lo ? hi - lo : 0;
  int32_t* cidx = chunk_idx + (size_t)unit * Kc;
  float* csc = chunk_score ? chunk_score + (size_t)unit * Kc : nullptr;
  // the pooled query of the unit, VPL consecutive values per lane (needed by the group stage: loaded early)
  constexpr int VPL = D / 32;
  float qf[VPL];
  if (Kg > 0) {
#pragma unroll
    for (int u = 0; u < VPL; ++u) qf[u] = q_pooled[(size_t)unit * D + lane * VPL + u];
  }

  // ---- stage the row (coalesced reads), pad with -inf -------------------------------------------------------
  HGA_RT_BEGIN;
  const int n_lanes = (n + m - 1) >> lm;  // lanes that own at least one candidate
  for (int c = lane; c < n_lanes * m; c += 32) {
    const float v = c < n ? row[lo + c] : -CUDART_INF_F;
    work[(c >> lm) * stride + (c & (m - 1))] = v;
  }
  __syncwarp();
  float* col = work + lane * stride;
  float bv = -CUDART_INF_F;
  int bo = 0;
  float v[M > 0 ? M : 1];
  if constexpr (M > 0) {
#pragma unroll
    for (int o = 0; o < M; o += 4) {
      const float4 t = lane < n_lanes ? *reinterpret_cast<const float4*>(col + o)
                                      : make_float4(-CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F);
      v[o] = t.x; v[o + 1] = t.y; v[o + 2] = t.z; v[o + 3] = t.w;
    }
    reg_rescan<M>(v, bv, bo);
  } else {
    if (lane < n_lanes) lane_rescan(col, m, bv, bo);
  }
  HGA_RT(16);

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
        if constexpr (M > 0) {
#pragma unroll
          for (int o = 0; o < M; ++o)
            if (o == bo) v[o] = -CUDART_INF_F;
          reg_rescan<M>(v, bv, bo);
        } else {
          col[bo] = -CUDART_INF_F;
          lane_rescan(col, m, bv, bo);
        }
      }
    }
  }
  HGA_RT(17);
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
  HGA_RT(18);

  // ---- group refinement: candidate `cand` = group cand % gpc of kept chunk cand / gpc (ascending group order) -----
  // Scores: one candidate per lane, fp64 fma chain over d (ascending) with the pooled query in shared memory as doubles.
  const int n_gc = cnt * gpc;  // <= 128
  const int gtake = min(Kg, n_gc);
  const bool need_scores = gtake < n_gc || group_score != nullptr;  // K_g >= candidates: every group is kept unscored
  __syncwarp();  // sel[] complete; the candidate rows in `work` are no longer needed
  HGA_RT(19);
  double* qd = reinterpret_cast<double*>(work);  // [D] the pooled query as doubles (the candidate rows are no longer needed)
  if (need_scores) {
#pragma unroll
    for (int u = 0; u < VPL; ++u) qd[lane * VPL + u] = (double)qf[u];
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
      gid[i] = g;
      gsc[i] = 0.f;
      if (!need_scores) continue;
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
  HGA_RT(20);
  unsigned taken = 0;  // bit i: candidate lane + 32*i is kept
  if (gtake == n_gc) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
      if (lane + 32 * i < n_gc) taken |= 1u << i;
  } else if (n_gc <= 64) {
    // at most two candidates per lane: rank every candidate against all others (value descending, index ascending) with 64
    // shuffles and keep the ranks below K_g -- one pass instead of K_g rounds of two warp reductions each
    const uint32_t k0 = lane < n_gc ? order_key(gsc[0]) : 0u;          // 0 is below the key of any float, -inf included
    const uint32_t k1 = lane + 32 < n_gc ? order_key(gsc[1]) : 0u;
    int r0 = 0, r1 = 0;  // candidates that come before candidate lane / lane + 32
#pragma unroll 8
    for (int sl = 0; sl < 32; ++sl) {
      const uint32_t a = __shfl_sync(kFull, k0, sl), b = __shfl_sync(kFull, k1, sl);  // candidates sl and sl + 32
      r0 += (a > k0 || (a == k0 && sl < lane)) ? 1 : 0;
      r0 += (b > k0) ? 1 : 0;                       // index sl + 32 > lane: a tie does not come before
      r1 += (a >= k1) ? 1 : 0;                      // index sl < lane + 32: a tie comes before
      r1 += (b > k1 || (b == k1 && sl < lane)) ? 1 : 0;
    }
    if (lane < n_gc && r0 < gtake) taken |= 1u;
    if (lane + 32 < n_gc && r1 < gtake) taken |= 2u;
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
  HGA_RT(21);
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
  HGA_RT(22);
#ifdef HGA_ROUTE_TRACE
  if (lane == 0) atomicAdd(&g_rt[31], 1ull);
#endif
}

}  // namespace

// One slab: the query blocks [d.jb, d.jb + d.nj), at most kRouteSlabRows of them; score_ws holds B * Hkv * d.nj rows.
static hga_status launch_route_slab(const Derived& d, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                                    int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                                    float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s) {
  const int nt = (d.n_b + kTile - 1) / kTile;
  dim3 grid(nt * (nt + 1) / 2, d.Hkv, d.B);
  score_kernel<<<grid, 128, 0, s>>>(q_pooled, chunk_sum, score_ws, d.n_b, d.D, d.F, d.L_eff, d.jb, d.jb + d.nj);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;

  const int n_units = d.B * d.Hkv * d.nj;
  const int kc_cap = d.Kc < d.n_b ? (d.Kc > 0 ? d.Kc : 1) : d.n_b;
  if (d.Kc <= 32 && kc_cap * d.gpc <= 128) {
    // fast path: register/redux rounds, one candidate per lane in the group stage
    const int n_max = d.n_b - d.F - d.L_eff > 1 ? d.n_b - d.F - d.L_eff : 1;
    int lm = 2;
    while ((32 << lm) < n_max) ++lm;
    const int per_warp_bytes = 32 * ((1 << lm) + 4) * 4 + 32 * 4;
    int warps = 4;
    while (warps > 1 && (size_t)warps * per_warp_bytes > 200 * 1024) warps >>= 1;
    const size_t smem = (size_t)warps * per_warp_bytes;
    if (smem <= 200 * 1024) {
      auto pick = [&](auto Dc) {
        constexpr int DD = decltype(Dc)::value;
        switch (lm) {
          case 4: return select_fast_kernel<DD, 16>;
          case 5: return select_fast_kernel<DD, 32>;
          default: return select_fast_kernel<DD, 0>;
        }
      };
      auto kern = d.D == 128 ? pick(std::integral_constant<int, 128>{}) : pick(std::integral_constant<int, 64>{});
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
                                                               d.n_g, d.gpc, d.F, d.L_eff, d.Kc, d.Kg, kc_cap, per_warp, 0, nullptr, nullptr);
  return launch_status();
}

// S2 + S3 over the query blocks [d.jb, d.jb + d.nj) in slabs of at most kRouteSlabRows blocks, one after the other on the
// stream: the score workspace is B * Hkv * min(n_b, kRouteSlabRows) rows of n_b floats (route_ws_rows), not n_b^2 per
// slice -- 16.8 MB at 64K tokens as before, 268 MB instead of 4.3 GB at 1 M tokens (B 1, H_kv 4); a decode step or a
// chunk append (hga_prefill_window) touches one row per slice.
hga_status launch_route(const Derived& d, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                        int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                        float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s, int slab_rows) {
  if (slab_rows <= 0 || slab_rows > kRouteSlabRows) slab_rows = kRouteSlabRows;
  for (int j0 = d.jb; j0 < d.jb + d.nj; j0 += slab_rows) {
    Derived ds = d;
    ds.jb = j0;
    ds.nj = d.jb + d.nj - j0 < slab_rows ? d.jb + d.nj - j0 : slab_rows;
    hga_status st = launch_route_slab(ds, q_pooled, chunk_sum, group_sum, chunk_idx, chunk_score, n_chunks, group_idx,
                                      group_score, n_groups, score_ws, s);
    if (st != HGA_OK) return st;
  }
  return HGA_OK;
}

}  // namespace hga (reopened below)

namespace hga {

namespace {

// ----------------------------------------------------------------------------------------------------------------
// N3 max rule on the tensor cores: approximate scores by a bf16 tcgen05 contraction, exact fp64 re-scoring of every
// candidate that can still belong to the top-K_c.
//   1. split_kernel        : S_c = hi + lo (two bf16 tables, |S_c - hi - lo| <= 2^-18 |S_c|) and |S_c|_2 per row;
//   2. score_max_tc_kernel : per (slice, block j): D[cand, row] = sum_d S_c[cand, d] q[row, d] for 128 candidates x the
//                            block's 64*G stored (bf16, exact) rotated queries, fp32 accumulation in TMEM, both bf16
//                            parts of S_c; the epilogue folds the rows with a max -> approximate score s~(j, cand);
//                            also q_max(j) = max_row |q_row|_2;
//   3. band_kernel         : tau = K_c-th largest s~ of the unit; every candidate whose s~ is within the error bound of
//                            tau (s~_c >= tau - E_max - e_c, e_c = eps |S_c|_2 q_max, eps = 2^-13 -- eight times the
//                            worst case of the two-part split plus fp32 accumulation over 2D products) is listed: the
//                            list provably contains the exact top-K_c;
//   4. score_max_kernel    : exact fp64 scores of the listed candidates (gathered mode); 5. the generic selection
//                            kernel's second phase picks the top-K_c of the list (ties -> lower index).
// A unit whose band does not fit the list (more than kBandCap candidates within the bound: degenerate, tied inputs) is
// flagged and recomputed by the dense fp64 path.
// ----------------------------------------------------------------------------------------------------------------
constexpr int kBandCap = 128;
constexpr float kBandEps = 1.0f / 8192.0f;  // 2^-13

template <int D>
__global__ void __launch_bounds__(128) split_kernel(const float* __restrict__ table, __nv_bfloat16* __restrict__ hi,
                                                    __nv_bfloat16* __restrict__ lo, float* __restrict__ norm, long long rows) {
  const long long row = (long long)blockIdx.x * 4 + threadIdx.x / 32;
  const int lane = threadIdx.x % 32;
  if (row >= rows) return;
  float ss = 0.f;
  for (int d = lane; d < D; d += 32) {
    const float v = table[row * D + d];
    const __nv_bfloat16 h = __float2bfloat16_rn(v);
    const __nv_bfloat16 l = __float2bfloat16_rn(v - __bfloat162float(h));
    hi[row * D + d] = h;
    lo[row * D + d] = l;
    ss = fmaf(v, v, ss);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, off);
  if (lane == 0) norm[row] = sqrtf(ss) * (1.0f + 1e-6f);  // rounded up: it enters an upper bound
}

template <int D>
struct TcS {
  static constexpr int kHalves = D / 64;
  static constexpr int kAHalf = 128 * 128;             // 128 candidates x 128 B
  static constexpr int kAPart = kHalves * kAHalf;      // one bf16 part (hi or lo) of the candidate tile
  static constexpr int kBHalf = 256 * 128;             // 256 query rows x 128 B
  static constexpr int kBBlk = kHalves * kBHalf;       // one block of up to 256 query rows
  static constexpr int kA = 0;
  static constexpr int kB = 2 * kAPart;
  static constexpr int kPairFlush = 128 * 32;          // (candidate, row) pairs one 32-column sweep can flag
  static constexpr int kPairCap = 2 * kPairFlush;      // the list is emptied once it holds more than kPairFlush
  // after the Q blocks: 3 mbarriers + the TMEM pointer (64 B), then the listed kernel's extras
  __host__ __device__ static constexpr int bars_off(int nblk) { return kB + nblk * kBBlk; }
  __host__ __device__ static constexpr int smem_bytes(int nblk) { return bars_off(nblk) + 64; }
  static constexpr int kExtra = 128 * 8 + 128 * 4 + 128 * 4 + 16 + kPairCap * 2;  // best keys, e_c, table rows, counter, pairs
  __host__ __device__ static constexpr int smem_bytes_listed(int nblk) { return smem_bytes(nblk) + kExtra; }
};

// Shared prologue of the two tensor-core kernels (all 128 threads): barriers, 512 TMEM columns, the block's queries
// (G heads x 64 rows, 4 heads per 256-row block) by TMA; returns the TMEM base once the queries are in shared memory.
template <int D>
__device__ __forceinline__ uint32_t tc_load_queries(unsigned char* smem, const CUtensorMap* tmQ, int G, long long qrow0, int N,
                                                    bool wait = true) {
  using namespace tc;
  using L = TcS<D>;
  const uint32_t sbase = smem_u32(smem);
  const int nblk = (G + 3) / 4;
  const uint32_t bars = sbase + (uint32_t)L::bars_off(nblk);  // [0] Q loaded, [1] A loaded, [2] MMAs done
  volatile uint32_t* tmem_p = reinterpret_cast<volatile uint32_t*>(smem + L::bars_off(nblk) + 32);
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();
    mbar_init(bars + 0, 1);
    mbar_init(bars + 8, 1);
    mbar_init(bars + 16, 1);
    fence_barrier_init();
    fence_proxy_async();
  }
  if (warp == 0) tmem_alloc(sbase + (uint32_t)(L::bars_off(nblk) + 32), 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_p;
  if (warp == 0) {
    if (lane == 0) mbar_expect_tx(bars + 0, (uint32_t)(64 * G * D * 2));
    __syncwarp();
    for (int i = lane; i < G * L::kHalves; i += 32) {
      const int h = i / L::kHalves, half = i % L::kHalves;
      tma_load_2d(sbase + (uint32_t)(L::kB + (h / 4) * L::kBBlk + half * L::kBHalf + (h % 4) * 64 * 128), tmQ, half * 64,
                  (int)(qrow0 + (long long)h * N), bars + 0);
    }
  }
  if (wait) mbar_wait(bars + 0, 0);  // otherwise the caller waits on barrier 0 (parity 0) before it reads the queries
  return tmem;
}

// max over the block's 64 G query rows of |q|_2, rounded up (it enters an error bound).  Eight lanes per row, one 16-byte
// piece each (a quarter-warp reads one whole 128-byte row: no bank conflicts); the swizzle permutes the pieces of a row,
// it does not mix rows.  Contains a __syncthreads.
template <int D>
__device__ __forceinline__ float tc_query_max_norm(const unsigned char* smem, int R, float* s_red) {
  using L = TcS<D>;
  float best = 0.f;
  const int sub = threadIdx.x % 8;
#pragma unroll 4
  for (int r = threadIdx.x / 8; r < R; r += 16) {
    float ss = 0.f;
#pragma unroll
    for (int half = 0; half < L::kHalves; ++half) {
      const uint4 v = *reinterpret_cast<const uint4*>(smem + L::kB + (r / 256) * L::kBBlk + half * L::kBHalf + (r % 256) * 128 + sub * 16);
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const float a0 = __uint_as_float(w[u] << 16), a1 = __uint_as_float(w[u] & 0xFFFF0000u);
        ss = fmaf(a0, a0, fmaf(a1, a1, ss));
      }
    }
    ss += __shfl_xor_sync(0xffffffffu, ss, 1);
    ss += __shfl_xor_sync(0xffffffffu, ss, 2);
    ss += __shfl_xor_sync(0xffffffffu, ss, 4);
    best = fmaxf(best, ss);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) best = fmaxf(best, __shfl_xor_sync(0xffffffffu, best, off));
  if (threadIdx.x % 32 == 0) s_red[threadIdx.x / 32] = best;
  __syncthreads();
  return sqrtf(fmaxf(fmaxf(s_red[0], s_red[1]), fmaxf(s_red[2], s_red[3]))) * (1.0f + 1e-5f);
}

// Warp 0, all lanes: D[cand, row] (TMEM, 128 lanes x 64 G columns) = (hi + lo)[cand, :] . q[row, :] for the candidate tile
// in shared memory; both bf16 parts accumulate into the same fp32 columns.  Commits to bars + 16.
template <int D>
__device__ __forceinline__ void tc_issue_tile(uint32_t sbase, uint32_t tmem, int G, uint32_t ld) {
  using namespace tc;
  using L = TcS<D>;
  constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);  // SBO 1024 B, version 1, SWIZZLE_128B
  constexpr uint32_t kLbo = (16u >> 4) << 16;
  const int nblk = (G + 3) / 4;
  for (int blk = 0; blk < nblk; ++blk) {
    const int nrows = 64 * min(4, G - 4 * blk);
    const uint32_t idesc = umma_idesc(128, nrows, false);
    const uint32_t d = tmem + (uint32_t)(blk * 256);
    const uint32_t bb = ((sbase + (uint32_t)(L::kB + blk * L::kBBlk)) & 0x3FFFFu) >> 4;
#pragma unroll
    for (int part = 0; part < 2; ++part) {
      const uint32_t ab = ((sbase + (uint32_t)(L::kA + part * L::kAPart)) & 0x3FFFFu) >> 4;
#pragma unroll
      for (int kk = 0; kk < D / 16; ++kk) {
        const uint32_t oa = (uint32_t)((kk / 4) * L::kAHalf + (kk % 4) * 32) >> 4;
        const uint32_t ob = (uint32_t)((kk / 4) * L::kBHalf + (kk % 4) * 32) >> 4;
        umma_ss_e(d, make_desc(ab + oa + kLbo, kDescHi), make_desc(bb + ob + kLbo, kDescHi), idesc, (part | kk) ? 1u : 0u, ld);
      }
    }
  }
  umma_commit_e(sbase + (uint32_t)L::bars_off(nblk) + 16, ld);
}

// This lane's (= candidate's) maximum over the block's query rows of the accumulator tile.
__device__ __forceinline__ float tc_row_max(uint32_t taddr, int G) {
  using namespace tc;
  float best = -CUDART_INF_F;
  const int nblk = (G + 3) / 4;
  for (int blk = 0; blk < nblk; ++blk) {
    const int nrows = 64 * min(4, G - 4 * blk);
    for (int c0 = 0; c0 < nrows; c0 += 32) {
      uint32_t v[32];
      tmem_ld32(taddr + (uint32_t)(blk * 256 + c0), v);
      tmem_wait_ld();
      float m0 = __uint_as_float(v[0]), m1 = __uint_as_float(v[1]);
#pragma unroll
      for (int c = 2; c < 32; c += 2) {
        m0 = fmaxf(m0, __uint_as_float(v[c]));
        m1 = fmaxf(m1, __uint_as_float(v[c + 1]));
      }
      best = fmaxf(best, fmaxf(m0, m1));
    }
  }
  return best;
}

template <int D>
__global__ void __launch_bounds__(128, 1)
score_max_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmHi,
                    const __grid_constant__ CUtensorMap tmLo, float* __restrict__ scores, float* __restrict__ qmax, int N, int n_b,
                    int G, int Hkv, int F, int L_eff, int jb) {
  using namespace tc;
  using L = TcS<D>;
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ float s_red[4];
  const uint32_t sbase = smem_u32(smem);
  const int j = jb + (int)blockIdx.x;
  const size_t slice = blockIdx.y;
  const size_t unit = slice * n_b + j;
  const int n_cand = j - L_eff;
  if (n_cand - F <= kBandCap) return;  // block-uniform: band_kernel lists every candidate of such a unit
  const int nblk = (G + 3) / 4;
  const uint32_t bars = sbase + (uint32_t)L::bars_off(nblk);
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int b = (int)(slice / Hkv), kv = (int)(slice % Hkv);
  const uint32_t ld = elect_one();  // meaningful in warp 0 only
  const uint32_t tmem = tc_load_queries<D>(smem, &tmQ, G, ((long long)b * Hkv * G + (long long)kv * G) * N + (long long)j * kChunk, N);
  {
    const float qm = tc_query_max_norm<D>(smem, 64 * G, s_red);
    if (threadIdx.x == 0) qmax[unit] = qm;
  }
  // ---- candidate tiles ---------------------------------------------------------------------------------------------------
  const int n_tiles = (n_cand + 127) / 128;
  const long long srow0 = (long long)slice * n_b;
  auto load_tile = [&](int a) {  // warp 0, all lanes: both bf16 parts of candidates [128 a, 128 a + 128)
    if (lane == 0) mbar_expect_tx(bars + 8, (uint32_t)(2 * L::kAPart));
    __syncwarp();
    if (lane < 2 * L::kHalves) {
      const int part = lane / L::kHalves, half = lane % L::kHalves;
      tma_load_2d(sbase + (uint32_t)(L::kA + part * L::kAPart + half * L::kAHalf), part == 0 ? &tmHi : &tmLo, half * 64,
                  (int)(srow0 + 128 * a), bars + 8);
    }
  };
  if (warp == 0) load_tile(0);
  for (int a = 0; a < n_tiles; ++a) {
    if (warp == 0) {
      mbar_wait(bars + 8, (uint32_t)a & 1u);
      tc_fence_after();
      tc_issue_tile<D>(sbase, tmem, G, ld);
    }
    mbar_wait(bars + 16, (uint32_t)a & 1u);
    tc_fence_after();
    if (warp == 0 && a + 1 < n_tiles) load_tile(a + 1);  // the MMAs have read the tile: the next one loads under the epilogue
    const float best = tc_row_max(tmem + ((uint32_t)(warp * 32) << 16), G);
    const int cand = 128 * a + warp * 32 + lane;
    if (cand < n_b) scores[unit * (size_t)n_b + cand] = best;
    tc_fence_before();
    __syncthreads();  // every lane has read its accumulator row; the candidate tile and TMEM may be overwritten
    tc_fence_after();
  }
  if (warp == 0) tmem_dealloc(tmem, 512);
}

__device__ __forceinline__ long long f64_key(double v) {  // order-preserving map of doubles onto signed integers
  const long long b = __double_as_longlong(v);
  return b >= 0 ? b : b ^ 0x7FFFFFFFFFFFFFFFll;
}

// Exact max-rule scores of LISTED candidates (the band of possible top-K_c chunks, or the group candidates of the kept
// chunks): out[unit][i] = max over the block's 64 G stored queries of <q, table row of candidate i> in fp64 (d ascending,
// one fma chain -- the same value score_max_kernel computes), found without scoring every (candidate, query) pair in
// fp64: the bf16 hi/lo tensor-core contraction gives every pair's score a~ with |a~ - a| <= e_c (e_c = eps |S_c| q_max,
// as in band_kernel); with m~ = max over queries of a~, the maximising query of the exact scores has a~ >= m~ - 2 e_c,
// so only the pairs within 2 e_c of their candidate's m~ (usually one) are re-scored exactly.
// Candidate i of a unit is table row  list[unit * list_stride + i / gpc] * gpc + i % gpc  (gpc = 1: the list holds rows).
template <int D>
__global__ void __launch_bounds__(128, 1)
score_max_listed_kernel(const __grid_constant__ CUtensorMap tmQ, const float* __restrict__ table, const int32_t* __restrict__ list, const int32_t* __restrict__ cnt,
                        float* __restrict__ out, int N, int n_b, int n_rows_tab, int G, int Hkv, int jb, int list_stride, int gpc,
                        int out_stride) {
  using namespace tc;
  using L = TcS<D>;
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ float s_red[4];
  const uint32_t sbase = smem_u32(smem);
  const int j = jb + (int)blockIdx.x;
  const size_t slice = blockIdx.y;
  const size_t unit = slice * n_b + j;
  const int n_l = cnt[unit] * gpc;
  if (n_l <= 0) return;  // block-uniform (also the units flagged -1 for the dense path)
  const int nblk = (G + 3) / 4;
  const int R = 64 * G;
  const uint32_t bars = sbase + (uint32_t)L::bars_off(nblk);
  unsigned char* extra = smem + L::smem_bytes(nblk);
  long long* best_key = reinterpret_cast<long long*>(extra);          // [128]
  float* s_norm = reinterpret_cast<float*>(extra + 128 * 8);          // [128] |S_c|_2 of the tile's candidates, rounded up
  int* trow = reinterpret_cast<int*>(extra + 128 * 8 + 128 * 4);      // [128] table row of the tile's candidates
  int* n_pairs = reinterpret_cast<int*>(extra + 128 * 8 + 128 * 8);   // pairs listed (degenerate path)
  uint16_t* pairs = reinterpret_cast<uint16_t*>(extra + 128 * 8 + 128 * 8 + 16);  // [kPairCap] (candidate << 9) | row
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int b = (int)(slice / Hkv), kv = (int)(slice % Hkv);
  const uint32_t ld = elect_one();
  HGA_RT_BEGIN;
  // the queries load (TMA) under the staging of the first candidate tile
  const uint32_t tmem = tc_load_queries<D>(smem, &tmQ, G, ((long long)b * Hkv * G + (long long)kv * G) * N + (long long)j * kChunk, N,
                                           false);
  HGA_RT(0);
  const float* S = table + slice * (size_t)n_rows_tab * D;
  const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16);
  const int n_tiles = (n_l + 127) / 128;
  const int me = warp * 32 + lane;  // this thread's candidate of a tile (its TMEM lane)
  float qm = 0.f;
  for (int a = 0; a < n_tiles; ++a) {
    // ---- stage the tile: fp32 rows -> bf16 hi + lo in the swizzled K-major layout, one warp per row, eight rows in
    // flight.  Dead rows keep whatever the tile held: their accumulator lanes are never read.
    const int n_live = min(128, n_l - 128 * a);
    {
      const int ci = 128 * a + me;
      trow[me] = me < n_live ? list[unit * list_stride + ci / gpc] * gpc + ci % gpc : -1;
      best_key[me] = f64_key(-CUDART_INF);
      if (me == 0) n_pairs[0] = 0;
    }
    __syncthreads();
    for (int i0 = warp; i0 < n_live; i0 += 32) {
      float4 v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int i = i0 + 4 * u;
        v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i < n_live && 4 * lane < D) v[u] = *reinterpret_cast<const float4*>(S + (size_t)trow[i] * D + 4 * lane);
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int i = i0 + 4 * u;
        if (i >= n_live) break;  // warp-uniform
        if (4 * lane < D) {
          const float f[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
          uint32_t h[2], l[2];
#pragma unroll
          for (int t = 0; t < 2; ++t) {
            const __nv_bfloat16 h0 = __float2bfloat16_rn(f[2 * t]), h1 = __float2bfloat16_rn(f[2 * t + 1]);
            const __nv_bfloat16 l0 = __float2bfloat16_rn(f[2 * t] - __bfloat162float(h0));
            const __nv_bfloat16 l1 = __float2bfloat16_rn(f[2 * t + 1] - __bfloat162float(h1));
            h[t] = (uint32_t)__bfloat16_as_ushort(h0) | ((uint32_t)__bfloat16_as_ushort(h1) << 16);
            l[t] = (uint32_t)__bfloat16_as_ushort(l0) | ((uint32_t)__bfloat16_as_ushort(l1) << 16);
          }
          const int half = (4 * lane) / 64, piece = ((4 * lane) % 64) / 8;  // 16-byte piece of the 128-byte row
          const int off = half * L::kAHalf + i * 128 + ((piece ^ (i % 8)) * 16) + (lane % 2) * 8;
          *reinterpret_cast<uint2*>(smem + L::kA + off) = make_uint2(h[0], h[1]);
          *reinterpret_cast<uint2*>(smem + L::kA + L::kAPart + off) = make_uint2(l[0], l[1]);
        }
        float ss = fmaf(v[u].x, v[u].x, fmaf(v[u].y, v[u].y, fmaf(v[u].z, v[u].z, v[u].w * v[u].w)));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
        if (lane == 0) s_norm[i] = sqrtf(ss) * (1.0f + 1e-5f);
      }
    }
    fence_proxy_async();  // the generic-proxy writes of the tile become visible to the tensor core
    HGA_RT(1);
    if (a == 0) {
      mbar_wait(bars + 0, 0);  // the queries
      qm = tc_query_max_norm<D>(smem, R, s_red);
    } else {
      __syncthreads();
    }
    HGA_RT(2);
    if (warp == 0) {
      tc_fence_after();
      tc_issue_tile<D>(sbase, tmem, G, ld);
    }
    mbar_wait(bars + 16, (uint32_t)a & 1u);
    tc_fence_after();
    HGA_RT(3);
    const bool live = me < n_live;
    const float thr = tc_row_max(taddr, G) - 2.0f * kBandEps * qm * s_norm[me];
    HGA_RT(4);
    // ---- second sweep: the pairs within the bound, re-scored exactly -------------------------------------------------
    // exact score of (candidate pc of the tile, query row r): fp64, d ascending, one fma chain
    auto exact_pair = [&](int pc, int r) -> double {
      const float* sp = S + (size_t)trow[pc] * D;
      const unsigned char* qb = smem + L::kB + (r / 256) * L::kBBlk + (r % 256) * 128;
      double acc = 0.0;
#pragma unroll 8
      for (int d0 = 0; d0 < D; d0 += 8) {
        const uint4 qv = *reinterpret_cast<const uint4*>(qb + (d0 / 64) * L::kBHalf + ((((d0 % 64) / 8) ^ (r % 8)) * 16));
        const float4 s0 = *reinterpret_cast<const float4*>(sp + d0), s1 = *reinterpret_cast<const float4*>(sp + d0 + 4);
        const uint32_t w[4] = {qv.x, qv.y, qv.z, qv.w};
        const float sv[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          acc = fma((double)__uint_as_float(w[u] << 16), (double)sv[2 * u], acc);
          acc = fma((double)__uint_as_float(w[u] & 0xFFFF0000u), (double)sv[2 * u + 1], acc);
        }
      }
      return acc;
    };
    // bit mask of the columns [col0, col0 + 32) of this lane's accumulator row that reach thr
    auto hits_of = [&](const uint32_t* v) -> uint32_t {
      // most 32-column steps hold no pair of this lane: one max tree decides that
      float m0 = max3(__uint_as_float(v[0]), __uint_as_float(v[1]), __uint_as_float(v[2]));
      float m1 = max3(__uint_as_float(v[3]), __uint_as_float(v[4]), __uint_as_float(v[5]));
#pragma unroll
      for (int c = 6; c < 30; c += 4) {
        m0 = max3(m0, __uint_as_float(v[c]), __uint_as_float(v[c + 1]));
        m1 = max3(m1, __uint_as_float(v[c + 2]), __uint_as_float(v[c + 3]));
      }
      m0 = max3(m0, __uint_as_float(v[30]), __uint_as_float(v[31]));
      uint32_t hit = 0;
      if (live && fmaxf(m0, m1) >= thr) {
        uint32_t h0 = 0, h1 = 0, h2 = 0, h3 = 0;
#pragma unroll
        for (int c = 0; c < 32; c += 4) {
          h0 |= (__uint_as_float(v[c]) >= thr ? 1u : 0u) << c;
          h1 |= (__uint_as_float(v[c + 1]) >= thr ? 1u : 0u) << (c + 1);
          h2 |= (__uint_as_float(v[c + 2]) >= thr ? 1u : 0u) << (c + 2);
          h3 |= (__uint_as_float(v[c + 3]) >= thr ? 1u : 0u) << (c + 3);
        }
        hit = (h0 | h1) | (h2 | h3);
      }
      return hit;
    };
    // Usual case: at most four query rows per candidate are within the bound; every lane keeps its own rows in
    // registers and re-scores them itself -- no list, no atomics, no barrier.
    int hr0 = 0, hr1 = 0, hr2 = 0, hr3 = 0, nh = 0;
    for (int blk = 0; blk < nblk; ++blk) {
      const int nrows = 64 * min(4, G - 4 * blk);
      for (int c0 = 0; c0 < nrows; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(taddr + (uint32_t)(blk * 256 + c0), v);
        tmem_wait_ld();
        uint32_t hit = hits_of(v);
        while (hit) {
          const int r = blk * 256 + c0 + __ffs(hit) - 1;
          hit &= hit - 1;
          if (nh == 0) hr0 = r;
          else if (nh == 1) hr1 = r;
          else if (nh == 2) hr2 = r;
          else if (nh == 3) hr3 = r;
          ++nh;
        }
      }
    }
    HGA_RT(5);
    if (!__syncthreads_or(nh > 4)) {
      if (live) {
        double best = exact_pair(me, hr0);  // nh >= 1: the row of the approximate maximum is always within the bound
        if (nh > 1) best = fmax(best, exact_pair(me, hr1));
        if (nh > 2) best = fmax(best, exact_pair(me, hr2));
        if (nh > 3) best = fmax(best, exact_pair(me, hr3));
        out[unit * (size_t)out_stride + 128 * a + me] = (float)best;
      }
    } else {
      // Degenerate inputs (many queries within the bound of the best, e.g. identical queries): (candidate, row) pairs go
      // to a shared list that all threads empty together whenever one more 32-column step might not fit.
      auto rescore = [&]() {  // all 128 threads; a barrier separates the list from the pushes
        const int np = n_pairs[0];
        for (int pi = threadIdx.x; pi < np; pi += 128) {
          const int pc = pairs[pi] >> 9, r = pairs[pi] & 511;
          atomicMax(&best_key[pc], f64_key(exact_pair(pc, r)));
        }
        __syncthreads();
        if (threadIdx.x == 0) n_pairs[0] = 0;
        __syncthreads();
      };
      for (int blk = 0; blk < nblk; ++blk) {
        const int nrows = 64 * min(4, G - 4 * blk);
        for (int c0 = 0; c0 < nrows; c0 += 32) {
          uint32_t v[32];
          tmem_ld32(taddr + (uint32_t)(blk * 256 + c0), v);
          tmem_wait_ld();
          uint32_t hit = hits_of(v);
          while (hit) {
            const int c = __ffs(hit) - 1;
            hit &= hit - 1;
            pairs[atomicAdd(&n_pairs[0], 1)] = (uint16_t)((me << 9) | (blk * 256 + c0 + c));
          }
          if (__syncthreads_or(*reinterpret_cast<volatile int*>(&n_pairs[0]) > L::kPairFlush)) rescore();  // block-uniform
        }
      }
      rescore();
      if (live) {
        const long long kb = best_key[me];
        out[unit * (size_t)out_stride + 128 * a + me] = (float)__longlong_as_double(kb >= 0 ? kb : kb ^ 0x7FFFFFFFFFFFFFFFll);
      }
    }
    HGA_RT(6);
    tc_fence_before();
    __syncthreads();  // the tile, its tables and TMEM are free for the next tile
    tc_fence_after();
  }
  if (warp == 0) tmem_dealloc(tmem, 512);
  HGA_RT(7);
#ifdef HGA_ROUTE_TRACE
  if (threadIdx.x == 0) atomicAdd(&g_rt[15], 1ull);
#endif
}

// One warp per unit: the candidates whose approximate score can still reach the top-K_c (see the block comment above).
__global__ void __launch_bounds__(128) band_kernel(const float* __restrict__ scores, const float* __restrict__ snorm,
                                                   const float* __restrict__ qmax, int32_t* __restrict__ band_list,
                                                   int32_t* __restrict__ band_cnt, int n_units, int jb, int nj, int n_b, int F,
                                                   int L_eff, int Kc, int per_warp_floats) {
  extern __shared__ __align__(16) float smem_f[];
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int widx = blockIdx.x * (blockDim.x / 32) + warp;
  if (widx >= n_units) return;
  float* work = smem_f + (size_t)warp * per_warp_floats;  // [n_b]
  const int j = jb + widx % nj;
  const size_t slice = widx / nj;
  const size_t unit = slice * n_b + j;
  const float* row = scores + unit * (size_t)n_b;
  const float* sn = snorm + slice * (size_t)n_b;
  const int lo = F, hi = j - L_eff;
  const int n = hi > lo ? hi - lo : 0;
  int32_t* list = band_list + unit * (size_t)kBandCap;
  if (n <= Kc || n <= kBandCap) {
    // every candidate is kept (n <= K_c) or fits the list anyway: exact scores for all of them
    const int m = min(n, kBandCap);
    for (int c = lane; c < m; c += 32) list[c] = lo + c;
    if (lane == 0) band_cnt[unit] = n <= kBandCap ? n : -1;
    return;
  }
  float snmax = 0.f;
  for (int c = lane; c < n; c += 32) {
    work[c] = row[lo + c];
    snmax = fmaxf(snmax, sn[lo + c]);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) snmax = fmaxf(snmax, __shfl_xor_sync(0xffffffffu, snmax, off));
  __syncwarp();
  warp_topk_mark(work, n, Kc, lane);  // the K_c best approximate scores become -inf in `work`
  float tau = CUDART_INF_F;
  for (int c = lane; c < n; c += 32)
    if (work[c] == -CUDART_INF_F) tau = fminf(tau, row[lo + c]);
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) tau = fminf(tau, __shfl_xor_sync(0xffffffffu, tau, off));
  const float qm = qmax[unit];
  const float e_max = kBandEps * qm * snmax;
  int cnt = 0;
  bool overflow = false;
  for (int c0 = 0; c0 < n; c0 += 32) {
    const int c = c0 + lane;
    const bool on = c < n && row[lo + c] >= tau - e_max - kBandEps * qm * sn[lo + c];
    const unsigned mk = __ballot_sync(0xffffffffu, on);
    const int pos = cnt + __popc(mk & ((1u << lane) - 1u));
    if (on && pos < kBandCap) list[pos] = lo + c;
    cnt += __popc(mk);
  }
  overflow = cnt > kBandCap;
  if (lane == 0) band_cnt[unit] = overflow ? -1 : cnt;
}

}  // namespace

// Workspace of the max rule, in floats: [B, Hkv, n_b, n_b] chunk scores | [B, Hkv, n_b, kc_cap * gpc] group-candidate
// scores | (tensor-core path) S_hi, S_lo bf16 [rows, D] | |S_c| [rows] | q_max [units] | band_list int32 [units, kBandCap]
// | band_cnt int32 [units] | band_score [units, kBandCap]; every part starts on a 256-byte boundary.
namespace {
struct MaxWs {
  size_t gscores, s_hi, s_lo, snorm, qmax, band_list, band_cnt, band_score, total;  // offsets in floats
};
inline size_t up64(size_t n) { return (n + 63) & ~(size_t)63; }
inline int max_kc_cap(const Derived& d) { return d.Kc < d.n_b ? (d.Kc > 0 ? d.Kc : 1) : d.n_b; }
inline MaxWs max_ws(const Derived& d) {
  MaxWs w;
  const size_t rows = (size_t)d.B * d.Hkv * d.n_b;
  size_t o = up64(rows * d.n_b);
  w.gscores = o; o += up64(rows * max_kc_cap(d) * d.gpc);
  w.s_hi = o; o += up64(rows * d.D / 2);
  w.s_lo = o; o += up64(rows * d.D / 2);
  w.snorm = o; o += up64(rows);
  w.qmax = o; o += up64(rows);
  w.band_list = o; o += up64(rows * kBandCap);
  w.band_cnt = o; o += up64(rows);
  w.band_score = o; o += up64(rows * kBandCap);
  w.total = o;
  return w;
}
// the tensor-core path: bf16 queries (exact operands), D in {64, 128}, the block's 64 G query rows in 512 TMEM columns
inline bool max_tc_eligible(const Derived& d) {
  return d.route_max == 1 && d.bf16_io && (d.D == 64 || d.D == 128) && d.G <= 8 && d.Kc > 0 && d.Kc <= 64 && d.n_b > kBandCap;
}
}  // namespace

size_t route_max_ws_bytes(const Derived& d) { return max_ws(d).total * sizeof(float); }

// N3 max rule: chunk scores (max over the block's stored rotated queries) -> top-K_c -> group candidate scores of the
// kept chunks -> top-K_g.
hga_status launch_route_max(const Derived& d, const void* q_rot, const float* chunk_sum, const float* group_sum,
                            int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                            float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s) {
  const int n_units = d.B * d.Hkv * d.nj;
  const int kc_cap = max_kc_cap(d);
  const MaxWs w = max_ws(d);
  float* gscores = score_ws + w.gscores;
  const bool use_tc = max_tc_eligible(d);
  const int per_warp = d.n_b + 2 * (use_tc && kBandCap > kc_cap * d.gpc ? kBandCap : kc_cap * d.gpc) + (use_tc ? kBandCap : kc_cap);
  int warps = 4;
  while (warps > 1 && (size_t)warps * per_warp * sizeof(float) > 200 * 1024) warps >>= 1;
  const size_t smem = (size_t)warps * per_warp * sizeof(float);
  if (smem > 200 * 1024) return HGA_ERR_UNSUPPORTED;
  auto sel = d.D == 128 ? select_generic_kernel<128> : select_generic_kernel<64>;
  HGA_CUDA_OK(cudaFuncSetAttribute(sel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int sel_grid = (n_units + warps - 1) / warps;
  const int ct = (d.n_b + kTile - 1) / kTile, gt = (kc_cap * d.gpc + kTile - 1) / kTile;
  // exact fp64 scores: dense over the chunk range (cidx == nullptr) or of the candidates listed in cidx / ncnt
  auto run_scores = [&](bool listed, const float* table, int n_rows_tab, const int32_t* cidx, const int32_t* ncnt, int list_cap,
                        int gpc, float* out, int out_stride, int tiles, const int32_t* only_neg) {
    dim3 grid(d.nj, tiles, d.B * d.Hkv);
    if (d.bf16_io)
      score_max_kernel<__nv_bfloat16><<<grid, 64, 0, s>>>((const __nv_bfloat16*)q_rot, table, cidx, ncnt, out, d.N, d.n_b, n_rows_tab,
                                                          d.D, d.G, d.Hkv, d.F, d.L_eff, d.jb, list_cap, gpc, out_stride, listed, only_neg);
    else
      score_max_kernel<float><<<grid, 64, 0, s>>>((const float*)q_rot, table, cidx, ncnt, out, d.N, d.n_b, n_rows_tab, d.D, d.G,
                                                  d.Hkv, d.F, d.L_eff, d.jb, list_cap, gpc, out_stride, listed, only_neg);
  };
  const int32_t* redo = nullptr;  // units the dense fp64 path still has to do (nullptr: all of them)
  CUtensorMap tmQ;
  // exact scores of listed candidates through the tensor-core row filter (score_max_listed_kernel)
  auto run_listed = [&](const float* table, int n_rows_tab, const int32_t* cidx, const int32_t* ncnt, int list_stride, int gpc,
                        float* out, int out_stride) -> bool {
    const int nblk = (d.G + 3) / 4;
    if (d.D == 128) {
      const int sm = TcS<128>::smem_bytes_listed(nblk);
      if (cudaFuncSetAttribute(score_max_listed_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return false;
      score_max_listed_kernel<128><<<dim3(d.nj, d.B * d.Hkv), 128, sm, s>>>(tmQ, table, cidx, ncnt, out, d.N, d.n_b, n_rows_tab, d.G,
                                                                           d.Hkv, d.jb, list_stride, gpc, out_stride);
    } else {
      const int sm = TcS<64>::smem_bytes_listed(nblk);
      if (cudaFuncSetAttribute(score_max_listed_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return false;
      score_max_listed_kernel<64><<<dim3(d.nj, d.B * d.Hkv), 128, sm, s>>>(tmQ, table, cidx, ncnt, out, d.N, d.n_b, n_rows_tab, d.G,
                                                                          d.Hkv, d.jb, list_stride, gpc, out_stride);
    }
    return cudaGetLastError() == cudaSuccess;
  };
  if (use_tc) {
    const long long rows = (long long)d.B * d.Hkv * d.n_b;
    __nv_bfloat16* s_hi = reinterpret_cast<__nv_bfloat16*>(score_ws + w.s_hi);
    __nv_bfloat16* s_lo = reinterpret_cast<__nv_bfloat16*>(score_ws + w.s_lo);
    float* snorm = score_ws + w.snorm;
    float* qmax = score_ws + w.qmax;
    int32_t* band_list = reinterpret_cast<int32_t*>(score_ws + w.band_list);
    int32_t* band_cnt = reinterpret_cast<int32_t*>(score_ws + w.band_cnt);
    float* band_score = score_ws + w.band_score;
    CUtensorMap tmHi, tmLo;
    if (!tc::make_map_2d(&tmQ, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, q_rot, (uint64_t)d.B * d.Hq * d.N, d.D, 64, 64) ||
        !tc::make_map_2d(&tmHi, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, s_hi, (uint64_t)rows, d.D, 64, 128) ||
        !tc::make_map_2d(&tmLo, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, s_lo, (uint64_t)rows, d.D, 64, 128))
      return HGA_ERR_CUDA;
    const int nblk = (d.G + 3) / 4;
    if (d.D == 128) {
      split_kernel<128><<<(unsigned)((rows + 3) / 4), 128, 0, s>>>(chunk_sum, s_hi, s_lo, snorm, rows);
      const int sm = TcS<128>::smem_bytes(nblk);
      HGA_CUDA_OK(cudaFuncSetAttribute(score_max_tc_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm));
      score_max_tc_kernel<128><<<dim3(d.nj, d.B * d.Hkv), 128, sm, s>>>(tmQ, tmHi, tmLo, score_ws, qmax, d.N, d.n_b, d.G, d.Hkv,
                                                                       d.F, d.L_eff, d.jb);
    } else {
      split_kernel<64><<<(unsigned)((rows + 3) / 4), 128, 0, s>>>(chunk_sum, s_hi, s_lo, snorm, rows);
      const int sm = TcS<64>::smem_bytes(nblk);
      HGA_CUDA_OK(cudaFuncSetAttribute(score_max_tc_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm));
      score_max_tc_kernel<64><<<dim3(d.nj, d.B * d.Hkv), 128, sm, s>>>(tmQ, tmHi, tmLo, score_ws, qmax, d.N, d.n_b, d.G, d.Hkv,
                                                                      d.F, d.L_eff, d.jb);
    }
    if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
    {
      int bw = 4;
      while (bw > 1 && (size_t)bw * d.n_b * sizeof(float) > 200 * 1024) bw >>= 1;
      const size_t bsm = (size_t)bw * d.n_b * sizeof(float);
      if (bsm > 200 * 1024) return HGA_ERR_UNSUPPORTED;
      HGA_CUDA_OK(cudaFuncSetAttribute(band_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
      band_kernel<<<(n_units + bw - 1) / bw, bw * 32, bsm, s>>>(score_ws, snorm, qmax, band_list, band_cnt, n_units, d.jb, d.nj,
                                                               d.n_b, d.F, d.L_eff, d.Kc, d.n_b);
    }
    if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
    // exact scores of the listed candidates, then the top-K_c of each list ("groups" of one chunk each)
    if (!run_listed(chunk_sum, d.n_b, band_list, band_cnt, kBandCap, 1, band_score, kBandCap)) return HGA_ERR_CUDA;
    sel<<<sel_grid, warps * 32, smem, s>>>(score_ws, nullptr, chunk_sum, band_list, nullptr, band_cnt, chunk_idx, chunk_score,
                                           n_chunks, n_units, d.jb, d.nj, d.n_b, d.n_b, 1, d.F, d.L_eff, kBandCap, d.Kc, kBandCap,
                                           per_warp, 2, band_score, nullptr);
    if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
    redo = band_cnt;  // units flagged -1: their band did not fit the list
  }
  run_scores(false, chunk_sum, d.n_b, nullptr, nullptr, d.Kc, d.gpc, score_ws, d.n_b, ct, redo);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
  sel<<<sel_grid, warps * 32, smem, s>>>(score_ws, nullptr, group_sum, chunk_idx, chunk_score, n_chunks, group_idx, group_score,
                                         n_groups, n_units, d.jb, d.nj, d.n_b, d.n_g, d.gpc, d.F, d.L_eff, d.Kc, d.Kg, kc_cap,
                                         per_warp, 1, nullptr, redo);
  if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
  if (d.Kg <= 0) return HGA_OK;
  if (use_tc) {
    if (!run_listed(group_sum, d.n_g, chunk_idx, n_chunks, d.Kc, d.gpc, gscores, kc_cap * d.gpc)) return HGA_ERR_CUDA;
  } else {
    run_scores(true, group_sum, d.n_g, chunk_idx, n_chunks, d.Kc, d.gpc, gscores, kc_cap * d.gpc, gt, nullptr);
    if (cudaGetLastError() != cudaSuccess) return HGA_ERR_CUDA;
  }
  sel<<<sel_grid, warps * 32, smem, s>>>(score_ws, nullptr, group_sum, chunk_idx, chunk_score, n_chunks, group_idx, group_score,
                                         n_groups, n_units, d.jb, d.nj, d.n_b, d.n_g, d.gpc, d.F, d.L_eff, d.Kc, d.Kg, kc_cap,
                                         per_warp, 2, gscores, nullptr);
  return launch_status();
}

// ----------------------------------------------------------------------------------------------------------------
// hga_route_static: S2 + S3 for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc) and have no workspace to pass.  The chunk-score matrix lives in a file-scope device array of
// HGA_ROUTE_STATIC_MAX_BYTES (16 MiB: BASELINE.json configs[4], B 1 x H_kv 4 x 1024 x 1024 floats, fits exactly); every
// GPU that loads the library holds it until the process exits.  In host code `g_route_static` is only the host-side
// stand-in of the symbol, never a device address: the address comes from cudaGetSymbolAddress, once per device with that
// device current.  No cudaMalloc / cudaFree / allocating library routine on this path.  All calls share the array, which
// keeps the previous call's contents; nothing has to start at zero (score_kernel writes every entry the selection kernels
// read, in the same call), but two calls that overlap on the GPU -- different streams, or graphs replayed concurrently --
// race on it.
// ----------------------------------------------------------------------------------------------------------------
namespace {
constexpr size_t kRouteStaticFloats = (size_t)HGA_ROUTE_STATIC_MAX_BYTES / sizeof(float);
static __device__ __align__(256) float g_route_static[kRouteStaticFloats];

constexpr int kMaxDevices = 64;
std::mutex g_route_static_mu;
float* g_route_static_ptr[kMaxDevices] = {};  // device address of g_route_static on device i (nullptr: not looked up yet)

// Device address of the scratch array on the current device; looked up once per device.
hga_status route_static_scratch(float** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return HGA_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_route_static_mu);
  if (g_route_static_ptr[dev] == nullptr) {
    float* ptr = nullptr;
    if (cudaGetSymbolAddress((void**)&ptr, g_route_static) != cudaSuccess || ptr == nullptr) {
      cudaGetLastError();  // leave no sticky-looking error behind for the caller's own checks
      return HGA_ERR_CUDA;
    }
    g_route_static_ptr[dev] = ptr;
  }
  *out = g_route_static_ptr[dev];
  return HGA_OK;
}
}  // namespace

hga_status launch_route_static(const Derived& d, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                               int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                               float* group_score, int32_t* n_groups, cudaStream_t s) {
  // the same B * Hkv * min(n_b, kRouteSlabRows) rows of n_b floats hga_route asks its caller for; larger problems are
  // refused, never truncated
  const size_t need = (size_t)d.B * d.Hkv * route_ws_rows(d.n_b) * d.n_b;
  if (need > kRouteStaticFloats) return HGA_ERR_WORKSPACE;
  float* scratch = nullptr;
  hga_status st = route_static_scratch(&scratch);
  if (st != HGA_OK) return st;
  return launch_route(d, q_pooled, chunk_sum, group_sum, chunk_idx, chunk_score, n_chunks, group_idx, group_score, n_groups,
                      scratch, s, 0);
}

}  // namespace hga

#ifdef HGA_ROUTE_TRACE
extern "C" __attribute__((visibility("default"))) void hga_debug_route_trace(unsigned long long* out) {
  cudaMemcpyFromSymbol(out, hga::g_rt, sizeof(unsigned long long) * 32);
}
#endif
