// S0 (RoPE on Q + pooled block query) and S1 (RoPE on K + mixed-RoPE chunk/group summaries).
// PAPER.md:62 (RoPE), 80-89 (summaries), 33/45/97 (chunk-shared per-KV-head routing query).
//
// One persistent, HBM-bound streaming kernel serves both stages (and both at once for hga_prefill):
//   * a tile = the 64 tokens x D elements of one (batch, head, chunk) -- contiguous in memory, 8..32 KB;
//   * every CTA owns a contiguous range of tiles, ordered (batch, chunk j) outermost; a consumer thread owns one
//     (token, 8 RoPE pairs) item of every tile, keeps its (cos, sin) in registers and recomputes them only when j
//     changes;
//   * a producer warp streams tiles global -> shared through a ring of bulk async copies (cp.async.bulk + mbarrier
//     complete_tx, full/empty barriers), so the bytes in flight per SM are set by the ring depth (128 KB), not by
//     registers or occupancy; consumers pull their 32 bytes into registers, release the stage at once, rotate and
//     write the result with 16-byte coalesced stores;
//   * a row (batch, j) holds Hkv K tiles followed by Hq Q tiles; a Q "unit" is the G heads of one KV group, whose
//     rotated values are pooled into the block's routing query; a K tile also yields its summaries.
//
// Numerics: the angle p*theta_i is reduced in fp64 (revolutions -> fractional part), the reduced angle is split
// into an fp32 head and tail, sincosf() is taken on the head and corrected to first order with the tail, so
// cos/sin carry ~1 ulp(fp32) error at any position.  The rotation is fp32 FMA.  Means are taken from the un-rounded
// fp32 values: per-thread / per-warp partial sums (at most 16 terms) in fp32 in a fixed order, combined in fp64
// and rounded once to float; the rotated tensor is rounded once (RNE) to io_dtype.
#include "hga_common.cuh"
#include "hga_tc_ptx.cuh"

namespace hga {

namespace {

using namespace tc;

constexpr int kMaxGpc = kChunk / 16;

__device__ __forceinline__ double reduced_angle(double pos, double turns) {
  double u = pos * turns;   // revolutions
  double fr = u - rint(u);  // [-0.5, 0.5]
  return fr * kTwoPi;
}

__device__ __forceinline__ float2 cos_sin_f32(double pos, double turns) {
  double ang = reduced_angle(pos, turns);
  float ah = (float)ang;
  float al = (float)(ang - (double)ah);
  float sh, ch;
  sincosf(ah, &sh, &ch);
  return make_float2(fmaf(-sh, al, ch), fmaf(ch, al, sh));
}

__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}

// 8 consecutive elements of a staged tile as fp32, through a 32-bit shared-space address (a generic pointer into the
// dynamic shared array makes ptxas re-derive the shared window base -- S2R SR_CgaCtaId + LEA -- at every tile)
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
  return r;
}
template <typename T>
__device__ __forceinline__ void load8_shared(uint32_t addr, float (&v)[8]);
template <>
__device__ __forceinline__ void load8_shared<float>(uint32_t addr, float (&v)[8]) {
  const uint4 a = lds128(addr), b = lds128(addr + 16);
  v[0] = __uint_as_float(a.x); v[1] = __uint_as_float(a.y); v[2] = __uint_as_float(a.z); v[3] = __uint_as_float(a.w);
  v[4] = __uint_as_float(b.x); v[5] = __uint_as_float(b.y); v[6] = __uint_as_float(b.z); v[7] = __uint_as_float(b.w);
}
template <>
__device__ __forceinline__ void load8_shared<__nv_bfloat16>(uint32_t addr, float (&v)[8]) {
  const uint4 r = lds128(addr);
  const uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    v[2 * i] = __uint_as_float(w[i] << 16);  // bf16 -> fp32 is exact
    v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
  }
}

struct RsParams {
  const void* q_raw;
  void* q_rot;    // nullable: skip the store
  float* pooled;  // nullable
  const void* k_raw;
  void* k_rot;       // nullable: skip the store
  float* chunk_sum;  // nullable
  float* group_sum;  // nullable
  int N, n_b;
  int jb, nj;     // query blocks / chunks [jb, jb + nj) are processed (hga_prefill_window)
  int tw0, tw1;   // token window: only rows t in [tw0, tw1) are stored and pooled; a chunk is summarised iff closed by tw1
  int HQ, PG;  // heads of the "Q" tensor (0: none), heads pooled together (a Q unit)
  int HK;      // heads of the "K" tensor (0: none)
  int gs, gpc, n_hi_c, n_hi_g;
  int tpr;     // tiles per row = HK + HQ
  long long pos0, pos_mod;
  long long total_tiles;  // rows * tpr
  // host-derived copies of per-tile tests (uniform; the 64-bit null tests and the power-of-two test were a measurable
  // share of the consumers' instruction stream): stores wanted, pooling wanted, PG - 1 when PG is a power of two else -1
  int store_q, store_k, pool_q, pg_mask;
};

// First tile of CTA `c` when `total` tiles are split over `n` CTAs at unit boundaries (a K tile, or PG Q tiles).
__device__ __forceinline__ long long range_start(long long c, long long n, const RsParams& p) {
  if (c >= n) return p.total_tiles;
  const long long raw = c * p.total_tiles / n;
  const long long row = raw / p.tpr;
  int r = (int)(raw % p.tpr);
  if (r > p.HK) r = p.HK + (r - p.HK + p.PG - 1) / p.PG * p.PG;
  return row * p.tpr + r;
}

template <typename T, int D>
struct RsCfg {
  static constexpr int kHalf = D / 2;
  static constexpr int kOct = D / 16;                // threads per token (8 pairs each)
  static constexpr int kConsumers = kChunk * kOct;   // one (token, 8 pairs) item per consumer thread
  static constexpr int kCWarps = kConsumers / 32;
  static constexpr int kThreads = kConsumers + 32;   // + the producer warp
  static constexpr int kTpw = 32 / kOct;             // tokens per consumer warp
  static constexpr int kCtasPerSm = (D == 128) ? 1 : 2;
  static constexpr int kTileBytes = kChunk * D * (int)sizeof(T);
  // shared memory map: fixed part first, the tile ring after it
  static constexpr int kPart = 0;                                        // [2][kCWarps][2][D] float
  static constexpr int kMid = kPart + 2 * kCWarps * 2 * D * 4;           // [2][kMaxGpc + 1][kHalf] double2
  static constexpr int kTurns = kMid + 2 * (kMaxGpc + 1) * kHalf * 16;   // [kHalf] double
  static constexpr int kBar = kTurns + kHalf * 8;                        // full[8], empty[8]
  static constexpr int kTiles = (kBar + 16 * 8 + 127) / 128 * 128;
  static constexpr int kBudget = (kCtasPerSm == 1 ? 200 : 100) * 1024;
  static constexpr int kStagesRaw = (kBudget - kTiles) / kTileBytes;
  static constexpr int kStages = kStagesRaw > 8 ? 8 : kStagesRaw;
  static constexpr int kBytes = kTiles + kStages * kTileBytes;
  static_assert(kStages >= 2, "ring too shallow");
};

__device__ __forceinline__ void consumer_sync(int n) { asm volatile("bar.sync 1, %0;" ::"r"(n) : "memory"); }

template <typename T, int D>
__global__ void __launch_bounds__(RsCfg<T, D>::kThreads, RsCfg<T, D>::kCtasPerSm)
rope_stream_kernel(const __grid_constant__ RopeFreq f, const __grid_constant__ RsParams p) {
  using C = RsCfg<T, D>;
  constexpr int half = C::kHalf, OCT = C::kOct, S = C::kStages, NW = C::kCWarps;
  extern __shared__ __align__(128) unsigned char smem[];
  uint32_t sbase = smem_u32(smem);
  // opaque to ptxas, which otherwise re-derives the shared-window base from SR_CgaCtaId (an S2R) at every barrier of every
  // tile (4 % of the kernel's stall samples on those S2R / LEA pairs)
  asm volatile("mov.u32 %0, %0;" : "+r"(sbase));
  float* part_base = reinterpret_cast<float*>(smem + C::kPart);
  double2* mid_base = reinterpret_cast<double2*>(smem + C::kMid);
  double* s_turns = reinterpret_cast<double*>(smem + C::kTurns);
  auto FULL = [&](int s) { return sbase + (uint32_t)C::kBar + 8u * (uint32_t)s; };
  auto EMPTY = [&](int s) { return sbase + (uint32_t)C::kBar + 64u + 8u * (uint32_t)s; };

  const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;

  const long long t0 = range_start(blockIdx.x, gridDim.x, p);
  const long long t1 = range_start((long long)blockIdx.x + 1, gridDim.x, p);
  const int nt = (int)(t1 - t0);

  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(FULL(s), 1);
      mbar_init(EMPTY(s), NW);
    }
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int i = tid; i < half; i += C::kThreads) s_turns[i] = f.turns[i];
  __syncthreads();

  // position of the CTA's first tile; every role advances (b, j, r) incrementally
  long long row0 = t0 / p.tpr;
  int r = (int)(t0 % p.tpr);
  int b = (int)(row0 / p.nj), j = p.jb + (int)(row0 % p.nj);

  if (warp == NW) {
    // ===================================== producer: bulk loads into the ring ===================================
    if (lane == 0) {
      for (int k = 0; k < nt; ++k) {
        const int s = k % S;
        if (k >= S) mbar_wait(EMPTY(s), (uint32_t)(k / S - 1) & 1u);
        const unsigned char* src;
        if (r < p.HK) src = (const unsigned char*)p.k_raw + (((size_t)b * p.HK + r) * p.N + (size_t)j * kChunk) * D * sizeof(T);
        else src = (const unsigned char*)p.q_raw + (((size_t)b * p.HQ + (r - p.HK)) * p.N + (size_t)j * kChunk) * D * sizeof(T);
        mbar_expect_tx(FULL(s), (uint32_t)C::kTileBytes);
        bulk_load(sbase + C::kTiles + s * C::kTileBytes, src, (uint32_t)C::kTileBytes, FULL(s));
        if (++r == p.tpr) {
          r = 0;
          if (++j == p.jb + p.nj) { j = p.jb; ++b; }
        }
      }
    }
    return;
  }
  // ======================================= consumers: rotate, store, reduce =====================================
  const int oct = tid % OCT, tok = tid / OCT;  // this thread's token of every tile, and its 8 pairs
  const int i0 = oct * 8;
  float2 tab[8];  // (cos, sin) of this thread's (token, pairs) for the current row
  float acc[16];
#pragma unroll
  for (int u = 0; u < 16; ++u) acc[u] = 0.f;
  bool fresh_row = true;
  int pb = 0;  // `part` buffer of the next reduction event (double buffered: one barrier per event)
  int mb = 1;  // `mid` buffer of the current row (flipped at every row change)

  for (int k = 0; k < nt; ++k) {
    const bool is_k = r < p.HK;
    if (fresh_row) {
      fresh_row = false;
      mb ^= 1;
      // chunk-aligned, and pos_mod is a multiple of the chunk: wrapping the chunk's first position wraps all 64
      long long pos_first = p.pos0 + (long long)j * kChunk;
      if (p.pos_mod > 0) pos_first %= p.pos_mod;
      const double pos = (double)(pos_first + tok);
#pragma unroll
      for (int u = 0; u < 8; ++u) tab[u] = cos_sin_f32(pos, s_turns[i0 + u]);
      if (p.HK > 0) {
        // middle positions (reading R2: start + (S-1)/2), full fp64 sincos; read after a K tile's barrier
        double2* mid = mid_base + mb * (kMaxGpc + 1) * half;
        for (int idx = tid; idx < (p.gpc + 1) * half; idx += C::kConsumers) {
          const int g = idx / half, i = idx - g * half;
          const double pm = (g < p.gpc) ? (double)pos_first + (double)(g * p.gs) + 0.5 * (double)(p.gs - 1)
                                        : (double)pos_first + 0.5 * (double)(kChunk - 1);
          double sn, cs;
          sincos(reduced_angle(pm, s_turns[i]), &sn, &cs);
          mid[idx] = make_double2(cs, sn);
        }
      }
    }
    const int s = k % S;
    mbar_wait(FULL(s), (uint32_t)(k / S) & 1u);
    const uint32_t rowa = sbase + (uint32_t)(C::kTiles + s * C::kTileBytes + (tok * D + i0) * (int)sizeof(T));
    float a[8], bb[8], ra[8], rb[8];
    load8_shared<T>(rowa, a);
    load8_shared<T>(rowa + half * (uint32_t)sizeof(T), bb);
    __syncwarp();
    if (lane == 0) mbar_arrive(EMPTY(s));  // the values are in registers: the stage can be refilled
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const float2 c = tab[u];
      ra[u] = fmaf(a[u], c.x, -(bb[u] * c.y));
      rb[u] = fmaf(bb[u], c.x, a[u] * c.y);
    }
    const int t_abs = j * kChunk + tok;
    const bool in_window = t_abs >= p.tw0 && t_abs < p.tw1;
    // store_q == 0: the rotated queries are only pooled (N2: S4 rotates its Q tiles itself)
    if ((is_k ? p.store_k : p.store_q) && in_window) {
      // token rows fit 32 bits (launch_stream checks B * heads * N < 2^31): one widening multiply per address
      T* base = is_k ? (T*)p.k_rot : (T*)p.q_rot;
      const int head = is_k ? b * p.HK + r : b * p.HQ + (r - p.HK);
      T* dst = base + (size_t)(unsigned)(head * p.N + t_abs) * D;
      Io<T>::store8(dst + i0, ra);
      Io<T>::store8(dst + half + i0, rb);
    }
    const bool pool = !is_k && p.pool_q;
    if (pool && in_window) {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        acc[u] += ra[u];
        acc[8 + u] += rb[u];
      }
    }
    // the runtime modulo is 25 instructions and was 12 % of the kernel's stall samples (ncu source page); G is a power of
    // two in every model shape of the paper
    const int q_done = r - p.HK + 1;
    const bool unit_end = pool && (p.pg_mask >= 0 ? (q_done & p.pg_mask) == 0 : q_done % p.PG == 0);
    float* part = part_base + (size_t)pb * NW * 2 * D;
    if (is_k) {
      // sums over the kTpw tokens of this warp (all inside one 16-token group), fixed order
#pragma unroll
      for (int u = 0; u < 8; ++u) {
#pragma unroll
        for (int off = OCT; off < 32; off <<= 1) {
          ra[u] += __shfl_xor_sync(0xffffffffu, ra[u], off);
          rb[u] += __shfl_xor_sync(0xffffffffu, rb[u], off);
          a[u] += __shfl_xor_sync(0xffffffffu, a[u], off);
          bb[u] += __shfl_xor_sync(0xffffffffu, bb[u], off);
        }
      }
      if (lane < OCT) {
        float* pr = part + (size_t)warp * 2 * D;  // [rot D][raw D]
        *reinterpret_cast<float4*>(pr + i0) = make_float4(ra[0], ra[1], ra[2], ra[3]);
        *reinterpret_cast<float4*>(pr + i0 + 4) = make_float4(ra[4], ra[5], ra[6], ra[7]);
        *reinterpret_cast<float4*>(pr + half + i0) = make_float4(rb[0], rb[1], rb[2], rb[3]);
        *reinterpret_cast<float4*>(pr + half + i0 + 4) = make_float4(rb[4], rb[5], rb[6], rb[7]);
        *reinterpret_cast<float4*>(pr + D + i0) = make_float4(a[0], a[1], a[2], a[3]);
        *reinterpret_cast<float4*>(pr + D + i0 + 4) = make_float4(a[4], a[5], a[6], a[7]);
        *reinterpret_cast<float4*>(pr + D + half + i0) = make_float4(bb[0], bb[1], bb[2], bb[3]);
        *reinterpret_cast<float4*>(pr + D + half + i0 + 4) = make_float4(bb[4], bb[5], bb[6], bb[7]);
      }
    } else if (unit_end) {
      // pooled query of the unit: reduce over the tokens of the warp, then (after the barrier) over the warps
#pragma unroll
      for (int u = 0; u < 16; ++u) {
#pragma unroll
        for (int off = OCT; off < 32; off <<= 1) acc[u] += __shfl_xor_sync(0xffffffffu, acc[u], off);
      }
      if (lane < OCT) {
        float* pr = part + (size_t)warp * D;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          pr[i0 + u] = acc[u];
          pr[half + i0 + u] = acc[8 + u];
        }
      }
#pragma unroll
      for (int u = 0; u < 16; ++u) acc[u] = 0.f;
    }
    if (is_k) {
      consumer_sync(C::kConsumers);
      pb ^= 1;
      const double2* mid = mid_base + mb * (kMaxGpc + 1) * half;
      for (int idx = tid; idx < (p.gpc + 1) * half; idx += C::kConsumers) {
        const int g = idx / half, i = idx - g * half;
        const bool chunk_level = g == p.gpc;
        const int span = chunk_level ? kChunk : p.gs;
        const int w0 = chunk_level ? 0 : g * p.gs / C::kTpw;
        const int w1 = chunk_level ? NW : (g + 1) * p.gs / C::kTpw;
        double sra = 0.0, srb = 0.0, swa = 0.0, swb = 0.0;
        for (int w = w0; w < w1; ++w) {  // warp w holds tokens [w*kTpw, (w+1)*kTpw)
          const float* pr = part + (size_t)w * 2 * D;
          sra += (double)pr[i];
          srb += (double)pr[half + i];
          swa += (double)pr[D + i];
          swb += (double)pr[D + half + i];
        }
        const double inv = 1.0 / (double)span;
        const int n_hi = chunk_level ? p.n_hi_c : p.n_hi_g;
        double sa, sb;
        if (i < n_hi) {  // high-frequency pair: rotate per token, then average
          sa = sra * inv;
          sb = srb * inv;
        } else {         // low-frequency pair: average raw keys, rotate at the middle position
          const double2 m = mid[idx];
          const double ma = swa * inv, mbv = swb * inv;
          sa = ma * m.x - mbv * m.y;
          sb = mbv * m.x + ma * m.y;
        }
        float* dstp = nullptr;
        if ((j + 1) * kChunk > p.tw1) {
          // the chunk is still open: only closed chunks are summarised
        } else if (chunk_level) {
          if (p.chunk_sum) dstp = p.chunk_sum + (((size_t)b * p.HK + r) * p.n_b + j) * D;
        } else if (p.group_sum) {
          dstp = p.group_sum + (((size_t)b * p.HK + r) * (size_t)(p.n_b * p.gpc) + (size_t)j * p.gpc + g) * D;
        }
        if (dstp) {
          dstp[i] = (float)sa;
          dstp[half + i] = (float)sb;
        }
      }
    } else if (unit_end) {
      consumer_sync(C::kConsumers);
      pb ^= 1;
      if (tid < D) {
        double sum = 0.0;
#pragma unroll
        for (int w = 0; w < NW; ++w) sum += (double)part[w * D + tid];
        const int n_pg = p.HQ / p.PG, pg = (r - p.HK) / p.PG;
        const int n_rows = min(p.tw1, (j + 1) * kChunk) - max(p.tw0, j * kChunk);  // rows of block j in the window
        p.pooled[(((size_t)b * n_pg + pg) * p.n_b + j) * D + tid] = (float)(sum / (double)(p.PG * n_rows));
      }
    }
    if (++r == p.tpr) {
      r = 0;
      fresh_row = true;
      if (++j == p.jb + p.nj) { j = p.jb; ++b; }
    }
  }
}

// N2 position tables for the in-kernel RoPE of S4: rope_a[j][i] = (cos, sin) of the first position of block j (wrapped like
// rope_stream_kernel wraps it), rope_b[t][i] = (cos, sin) of offset t, both with cos_sin_f32's accuracy; the angle of
// token 64 j + t is their sum, so S4 needs 512 bytes per block plus one 64-row table that stays in L1.
__global__ void rope_tables_kernel(const __grid_constant__ RopeFreq f, float2* __restrict__ rope_a, float2* __restrict__ rope_b,
                                   int n_b, int half, long long pos0, long long pos_mod) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_a = n_b * half;
  if (idx < n_a) {
    const int j = idx / half, i = idx % half;
    long long pos_first = pos0 + (long long)j * kChunk;
    if (pos_mod > 0) pos_first %= pos_mod;
    rope_a[idx] = cos_sin_f32((double)pos_first, f.turns[i]);
  } else if (idx < n_a + kChunk * half) {
    const int t = (idx - n_a) / half, i = (idx - n_a) % half;
    rope_b[idx - n_a] = cos_sin_f32((double)t, f.turns[i]);
  }
}

template <typename T, int D>
hga_status launch_stream_t(const RopeFreq& f, RsParams p, long long rows, cudaStream_t s) {
  using C = RsCfg<T, D>;
  const int n_sm = current_sm_count();
  if (n_sm <= 0) return HGA_ERR_CUDA;
  p.tpr = p.HK + p.HQ;
  p.total_tiles = rows * p.tpr;
  p.store_q = p.q_rot != nullptr;
  p.store_k = p.k_rot != nullptr;
  p.pool_q = p.pooled != nullptr;
  p.pg_mask = (p.PG & (p.PG - 1)) == 0 ? p.PG - 1 : -1;
  const long long units = rows * (p.HK + (p.HQ ? p.HQ / p.PG : 0));
  const int ctas_per_sm = C::kCtasPerSm;
  const long long cap = (long long)n_sm * ctas_per_sm;
  const int grid = (int)(units < cap ? units : cap);
  if (grid <= 0) return HGA_OK;
  auto kern = rope_stream_kernel<T, D>;
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::kBytes));
  kern<<<grid, C::kThreads, C::kBytes, s>>>(f, p);
  return launch_status();
}

hga_status launch_stream(const Derived& d, const RopeFreq& f, const RsParams& p, cudaStream_t s) {
  const long long rows = (long long)d.B * d.nj;
  if ((long long)d.B * (p.HQ > p.HK ? p.HQ : p.HK) * d.N >= (1ll << 31)) return HGA_ERR_UNSUPPORTED;  // 32-bit token rows
  if (d.bf16_io) {
    return d.D == 128 ? launch_stream_t<__nv_bfloat16, 128>(f, p, rows, s) : launch_stream_t<__nv_bfloat16, 64>(f, p, rows, s);
  }
  return d.D == 128 ? launch_stream_t<float, 128>(f, p, rows, s) : launch_stream_t<float, 64>(f, p, rows, s);
}

RsParams base_params(const Derived& d) {
  RsParams p = {};
  p.N = d.N; p.n_b = d.n_b;
  p.jb = d.jb; p.nj = d.nj; p.tw0 = (int)d.tw0; p.tw1 = (int)d.tw1;
  p.PG = 1;
  p.gs = d.gs; p.gpc = d.gpc; p.n_hi_c = d.n_hi_c; p.n_hi_g = d.n_hi_g;
  p.pos0 = d.pos0;
  p.pos_mod = d.pos_mod;
  return p;
}

}  // namespace

// S0 + S1 in one launch (hga_prefill): K tiles and Q tiles of a row share the position tables.
hga_status launch_rope_summaries(const Derived& d, const RopeFreq& f, const void* q_raw, void* q_rot, float* pooled,
                                 const void* k_raw, void* k_rot, float* chunk_sum, float* group_sum, cudaStream_t s) {
  RsParams p = base_params(d);
  p.q_raw = q_raw; p.q_rot = q_rot; p.pooled = pooled;
  p.HQ = d.Hq; p.PG = pooled ? d.G : 1;
  p.k_raw = k_raw; p.k_rot = k_rot; p.chunk_sum = chunk_sum; p.group_sum = group_sum;
  p.HK = d.Hkv;
  return launch_stream(d, f, p, s);
}

hga_status launch_rope_tables(const Derived& d, const RopeFreq& f, float2* rope_a, float2* rope_b, cudaStream_t s) {
  const int half = d.D / 2, total = (d.n_b + kChunk) * half;
  rope_tables_kernel<<<(total + 255) / 256, 256, 0, s>>>(f, rope_a, rope_b, d.n_b, half, d.pos0, d.pos_mod);
  return launch_status();
}

hga_status launch_rope(const Derived& d, const RopeFreq& f, const void* x_raw, int n_heads, void* x_rot, float* pooled,
                       cudaStream_t s) {
  RsParams p = base_params(d);
  p.q_raw = x_raw; p.q_rot = x_rot; p.pooled = pooled;
  p.HQ = n_heads; p.PG = pooled ? n_heads / d.Hkv : 1;
  return launch_stream(d, f, p, s);
}

hga_status launch_summaries(const Derived& d, const RopeFreq& f, const void* k_raw, void* k_rot, float* chunk_sum,
                            float* group_sum, cudaStream_t s) {
  RsParams p = base_params(d);
  p.k_raw = k_raw; p.k_rot = k_rot; p.chunk_sum = chunk_sum; p.group_sum = group_sum;
  p.HK = d.Hkv;
  return launch_stream(d, f, p, s);
}

}  // namespace hga
