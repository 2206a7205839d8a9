// S4, persistent tensor-core kernel for bf16 inputs (Eq. (1) PAPER.md:56 over the union set).
//
// One CTA per SM loops over work items; an item = one (batch, kv head, query block j) unit x two 128-row query
// tiles (a tile = 2 query heads of the GQA group x 64 tokens).  Every role runs the same item sequence and the
// roles are decoupled by mbarriers only, so the pipeline never drains between items: while the softmax
// warpgroups finish item n, the producer already gathers item n+1's keys, the tensor pipe starts its first
// Q K^T, and the epilogue warpgroup drains item n's output.
//
//   warps 0-3 / 4-7  softmax warpgroups (query tile 0 / 1), one thread per query row, ping-pong on the tensor pipe
//   warps 8-11       epilogue: O_t / l -> swizzled staging tile -> TMA store
//   warp 12          tcgen05.mma issuer (one thread):  S_t = Q_t K^T (SS),  O_t += P_t V (TS, P_t bf16 in TMEM)
//   warp 13          TMA producer: gathers the K and V pieces of the key list (16 rows x 64 bf16 boxes, 128B swizzle)
//   warp 14          key-list builder for the next item (double buffered)
//
// P_t is handed to the tensor pipe in two halves (keys 0..63 while 64..127 are still being exponentiated), which takes
// half a P V off the tile's softmax -> P V -> Q K^T latency chain.
//
// Split mode (template kSplit; G <= 2, i.e. one query tile per item): the tile runs on BOTH softmax warpgroups --
// virtual tile t owns (S_t, O_t) and the key tiles t, t+2, ... -- so two chains overlap on the tensor pipe as in the
// general case; the epilogue merges the two partial (m, l, O) results.  kPad (odd G, G = 1): softmax warps whose 32
// rows belong to the padding head skip the arithmetic and only keep the barrier sequence.
//
// Key order inside an item: current chunk first (so the causal mask lives only in columns 0..63 of tile 0), then
// sink chunks, routed groups, local chunks; only the last 128-key tile can be partial.
// TMEM map (512 columns): S_t at t*128 (P_t overlays its first 64 columns), O_t at 256 + t*D.
//
// Softmax arithmetic: fp32, base-2 (scores scaled by scale*log2 e), running max refreshed lazily (only when it grows
// by more than 2^8, which leaves the result mathematically unchanged), packed FFMA2/FADD2, FMNMX3 row max.
// A share of the exponentials CAN be evaluated on the FMA pipe (Cody-Waite + degree-3 polynomial, rel. error
// 7.5e-5, far below the bf16 rounding of P; HGA_S4_EMU_COUNT of every HGA_S4_EMU_PERIOD pairs).  It is off by
// default: the softmax step sits on the latency chain softmax -> P V -> Q K^T -> softmax of its tile, and ncu shows
// that chain bound by the warpgroup's instruction count, not by MUFU.EX2 throughput (XU pipe 43 % busy), so the
// ~6 extra instructions per emulated element cost more than the MUFU slot they free.
#include <cuda.h>
#include <math_constants.h>

#include <type_traits>

#include "hga_attend_softmax.cuh"
#include "hga_common.cuh"
#include "hga_tc_ptx.cuh"

namespace hga {

namespace {

using namespace tc;

constexpr int kThreads = 512;
constexpr int kEpiWarp0 = 8;
constexpr int kMmaWarp = 12;
constexpr int kLoadWarp = 13;
constexpr int kListWarp = 14;
constexpr int kTileKeys = 128;  // keys per KV tile (8 pieces of 16)
constexpr int kPPT = 8;         // pieces per tile
constexpr int kRegsSoftmax = 200, kRegsEpi = 64, kRegsCtl = 48;  // 2*128*200 + 128*64 + 128*48 = 65536

#ifdef HGA_S4_TRACE
__device__ long long g_trace[4096];
#define HGA_TRM(slot) do { if (tron && lane == 0) g_trace[slot] = clock64(); } while (0)
#else
#define HGA_TRM(slot) do { } while (0)
#endif

struct Tc2Params {
  int B, Hq, Hkv, N, n_b, G;
  int jb, nj;  // query blocks [jb, jb + nj) of every (batch, kv head) are processed
  int F, L_eff, gs, Kg;
  int n_mt;           // 128-row query tiles per unit = ceil(G/2)
  int ctas_per_unit;  // ceil(n_mt/2)
  int split;          // n_mt == 1 (G <= 2): the single query tile runs on both softmax warpgroups, key tiles split even/odd
  int list_cap;       // pieces per list buffer
  int n_items;
  float scale_log2;   // softmax_scale * log2(e)
  int out_bf16;
  // kRawQ (N2, the Q_rot round trip removed): tmQ maps the UN-rotated queries and the epilogue warpgroup rotates every Q
  // tile in shared memory before its first Q K^T.  (cos, sin) of position pos0 + 64 j + t for pair i is the product of
  // rope_a[j][i] (the block's first position) and rope_b[t][i] (offset t inside the block), both from launch_rope_tables.
  const float2* rope_a;  // [n_b][D/2]
  const float2* rope_b;  // [64][D/2]
};

template <int D>
struct Smem2 {
  static constexpr int kHalves = D / 64;                   // 64-element (128-byte) column blocks
  static constexpr int kHalfBytes = kTileKeys * 128;       // 128 rows x 128 B = 16 KB
  static constexpr int kTileBytes = kHalves * kHalfBytes;  // Q tile / K tile / V tile
  static constexpr int kStages = (D == 128) ? 2 : 4;
  static constexpr int kQ = 0;
  static constexpr int kK = kQ + 2 * kTileBytes;
  static constexpr int kV = kK + kStages * kTileBytes;
  static constexpr int kStage = kV + kStages * kTileBytes;  // epilogue staging: 4 warps x 4 KB
  static constexpr int kBar = kStage + 4 * 4096;
  // barrier ids
  static constexpr int QFULL = 0, QEMPTY = 2, SFULL = 4, PFULL = 6, OFULL = 8, OEMPTY = 10, LFULL = 12, LEMPTY = 14,
                       LISTFULL = 16, LISTEMPTY = 18, KFULL = 20, KEMPTY = KFULL + kStages, VFULL = KEMPTY + kStages,
                       VEMPTY = VFULL + kStages, PFULLB = VEMPTY + kStages, QROT = PFULLB + 2, kNumBars = QROT + 2;
  static constexpr int kMisc = kBar + 8 * kNumBars;  // tmem base (4 B), n_pieces[2]
  static constexpr int kInvL = kMisc + 16;           // 2 tiles x 128 rows fp32: 1/l (split mode: l), then m (split mode)
  static constexpr int kList = kInvL + 4 * 128 * 4;  // 2 x list_cap ints
};

struct Item {
  int b, kv, j, mt0, nt;
};

__device__ __forceinline__ Item decode_item(int it, const Tc2Params& prm) {
  // (batch, kv head) outermost: the K/V of one head (c5: 33.5 MB) then stays L2-resident while Q streams through,
  // and the CTAs working at any moment share sink / routed / local lines.  Inside a head: j descending (longest
  // lists first, the short early blocks fill the tail), the CTAs of one unit adjacent.
  const int per_head = prm.nj * prm.ctas_per_unit;
  Item r;
  const int bk = it / per_head;
  const int rem = it % per_head;
  r.j = prm.jb + prm.nj - 1 - rem / prm.ctas_per_unit;
  const int cu = rem % prm.ctas_per_unit;
  r.kv = bk % prm.Hkv;
  r.b = bk / prm.Hkv;
  r.mt0 = cu * 2;
  r.nt = min(2, prm.n_mt - r.mt0);
  return r;
}

// kSplit: one query tile per item (G <= 2), see the MMA issuer.  kPad: some tile holds a padding head (odd G).
template <int D, bool kSplit, bool kPad, bool kRawQ>
__global__ void __launch_bounds__(kThreads, 1)
attend_tc2_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                  const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmO,
                  const int32_t* __restrict__ group_idx, float* __restrict__ lse, const Tc2Params prm) {
  using L = Smem2<D>;
  extern __shared__ __align__(1024) unsigned char smem[];
  const uint32_t sbase = smem_u32(smem);
  auto BAR = [&](int i) { return sbase + (uint32_t)L::kBar + 8u * (uint32_t)i; };
  volatile uint32_t* tmem_base_p = reinterpret_cast<volatile uint32_t*>(smem + L::kMisc);
  volatile int* s_np = reinterpret_cast<volatile int*>(smem + L::kMisc + 4);  // [2]
  float* s_invl = reinterpret_cast<float*>(smem + L::kInvL);                  // [2][128]
  float* s_m = s_invl + 2 * 128;                                              // [2][128], split mode only
  int* s_list = reinterpret_cast<int*>(smem + L::kList);                      // [2][list_cap]

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();  // the 128B-swizzled tiles need a 1024-byte aligned base
    for (int t = 0; t < 2; ++t) {
      mbar_init(BAR(L::QFULL + t), 1);
      mbar_init(BAR(L::QEMPTY + t), 1);
      mbar_init(BAR(L::QROT + t), 4);  // the four epilogue warps, after rotating the tile (kRawQ)
      mbar_init(BAR(L::SFULL + t), 1);
      mbar_init(BAR(L::PFULL + t), 4);
      mbar_init(BAR(L::PFULLB + t), 4);
      mbar_init(BAR(L::OFULL + t), 1);
      mbar_init(BAR(L::OEMPTY + t), 4);
      mbar_init(BAR(L::LFULL + t), 4);
      mbar_init(BAR(L::LEMPTY + t), 4);
      mbar_init(BAR(L::LISTFULL + t), 1);
      mbar_init(BAR(L::LISTEMPTY + t), 10);  // producer + MMA + 8 softmax warps
    }
    for (int s = 0; s < L::kStages; ++s) {
      mbar_init(BAR(L::KFULL + s), 1);
      mbar_init(BAR(L::KEMPTY + s), 1);
      mbar_init(BAR(L::VFULL + s), 1);
      mbar_init(BAR(L::VEMPTY + s), 1);
    }
    fence_barrier_init();
    fence_proxy_async();
  }
  if (warp == kMmaWarp) tmem_alloc(sbase + L::kMisc, 512);
  if (warp == kLoadWarp && lane == 0) {
    prefetch_tmap(&tmQ);
    prefetch_tmap(&tmK);
    prefetch_tmap(&tmV);
  }
  if (warp == kEpiWarp0 && lane == 0) prefetch_tmap(&tmO);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_base_p;

  if (warp < 8) {
    // ===================================== softmax warpgroups ===================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsSoftmax));
    const int t = warp / 4;
    const int row = (warp % 4) * 32 + lane;  // row of the 128-row tile == TMEM lane
    const int r64 = row % 64;
    const uint32_t lane_base = (uint32_t)((warp % 4) * 32) << 16;
    const uint32_t s_addr = tmem + lane_base + (uint32_t)(t * 128);
    const uint32_t o_addr = tmem + lane_base + (uint32_t)(256 + t * D);
    const float sl2 = prm.scale_log2;
    uint32_t s_cnt = 0;  // S_FULL completions consumed
    uint32_t n_done = 0; // items this warpgroup has processed
    int k = 0;
    for (int it = blockIdx.x; it < prm.n_items; it += gridDim.x, ++k) {
      const Item im = decode_item(it, prm);
      const int buf = k & 1;
      mbar_wait(BAR(L::LISTFULL + buf), (uint32_t)(k >> 1) & 1u);
      const int n_pieces = s_np[buf];
      __syncwarp();
      if (lane == 0) mbar_arrive(BAR(L::LISTEMPTY + buf));
      constexpr bool split = kSplit;
      if (!split && t >= im.nt) continue;
      const int n_tiles = (n_pieces + kPPT - 1) / kPPT;
      float m_run = -CUDART_INF_F;  // running reference max, raw logit units
      float l_run = 0.f;
      // split mode: this warpgroup takes key tiles t, t+2, ... of the item's single query tile; the two partial
      // (m, l, O) results are merged by the epilogue warpgroup
      const int i_first = split ? t : 0, i_step = split ? 2 : 1;
      const bool dead = (kDiag & 1) || kPad && (im.mt0 + (split ? 0 : t)) * 2 + row / 64 >= prm.G;  // warp-uniform: a warp is 32 rows of one head
      for (int i = i_first; i < n_tiles; i += i_step) {
        const int nk = min(kPPT, n_pieces - i * kPPT) * 16;  // valid key columns of this tile
        mbar_wait(BAR(L::SFULL + t), s_cnt & 1u);
        ++s_cnt;
        if (dead) {
          // rows of a padding head (odd G, G = 1): nothing is stored from them, so no softmax either -- P stays
          // whatever it was and only feeds O rows that are never read.  The wait above keeps the warp in step
          // with the tile sequence (the next S arrives only after this tile's P barrier has completed).
          __syncwarp();
          if (lane == 0) {
            mbar_arrive(BAR(L::PFULL + t));
            mbar_arrive(BAR(L::PFULLB + t));
          }
          continue;
        }
        long long* tr = nullptr;
#ifdef HGA_S4_TRACE
        if (blockIdx.x == 0 && k >= 8 && k < 10 && (warp % 4) == 0 && i < 8) {
          tr = g_trace + (((k - 8) * 8 + i) * 2 + t) * 8;
          if (lane == 0) tr[0] = clock64();
        }
#endif
        tc_fence_after();
        softmax_tile<D>(
            s_addr, o_addr, i == 0, r64, nk, i != i_first, sl2, m_run, l_run,
            [&] {
              __syncwarp();
              if (lane == 0) mbar_arrive(BAR(L::PFULL + t));
            },
            [&] {
              __syncwarp();
              if (lane == 0) mbar_arrive(BAR(L::PFULLB + t));
            },
            tr);
      }
      // ---- item done: hand 1/l to the epilogue warpgroup, write LSE ----------------------------------------------
      mbar_wait(BAR(L::LEMPTY + t), (n_done & 1u) ^ 1u);
      ++n_done;
      s_invl[t * 128 + row] = split ? l_run : 1.f / l_run;
      if (split) s_m[t * 128 + row] = m_run * sl2;  // log2 units; -inf when this half saw no key tile
      const int head_in_group = (im.mt0 + t) * 2 + row / 64;
      if (!split && lse != nullptr && head_in_group < prm.G) {
        const size_t orow = ((size_t)im.b * prm.Hq + (size_t)(im.kv * prm.G + head_in_group)) * prm.N + (size_t)im.j * kChunk + r64;
        lse[orow] = (m_run * sl2 + log2f(l_run)) * 0.69314718055994530942f;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(BAR(L::LFULL + t));
    }
  } else if (warp < kMmaWarp) {
    // ===================================== epilogue warpgroup ===================================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsEpi));
    const int e = warp - kEpiWarp0;  // TMEM lanes 32e .. 32e+31
    const uint32_t lane_base = (uint32_t)(e * 32) << 16;
    const uint32_t stage = sbase + (uint32_t)L::kStage + (uint32_t)e * 4096u;
    unsigned char* stage_p = smem + L::kStage + e * 4096;
    const int colw = prm.out_bf16 ? 64 : 32;  // columns per 128-byte staging row
    uint32_t o_cnt[2] = {0, 0};  // items drained per tile
    const uint64_t pol_o = policy_evict_first();
    // kRawQ: RoPE on the Q tiles of an item, in place in shared memory, as soon as the raw tile has landed (during the
    // previous item's last key-tile step, when this warpgroup is idle) and before the issuer's first Q K^T of the tile.
    // A thread takes (token, 8 pairs) of both heads of the tile: x = columns [8 pc, 8 pc + 8), y = the same + D/2; the
    // arithmetic is rope_stream_kernel's (fp32 FMA, one RNE rounding to bf16).
    uint32_t qr_cnt[2] = {0, 0};  // Q tiles rotated per slot
    auto rotate_item = [&](const Item& im) {
      constexpr int PCS = D / 16;  // 8-pair pieces per row
      const int eid = e * 32 + lane;
      for (int t = 0; t < (kSplit ? 2 : im.nt); ++t) {
        mbar_wait(BAR(L::QFULL + t), qr_cnt[t] & 1u);
        ++qr_cnt[t];
        unsigned char* qt = smem + L::kQ + t * L::kTileBytes;
        const float2* ta = prm.rope_a + (size_t)im.j * (D / 2);
        for (int task = eid; task < 64 * PCS; task += 128) {
          const int tok = task / PCS, pc = task % PCS;
          float2 cs[8];
#pragma unroll
          for (int h4 = 0; h4 < 2; ++h4) {
            const float4* pa = reinterpret_cast<const float4*>(ta + pc * 8 + h4 * 4);
            const float4* pb = reinterpret_cast<const float4*>(prm.rope_b + (size_t)tok * (D / 2) + pc * 8 + h4 * 4);
            const float4 a01 = __ldg(pa), a23 = __ldg(pa + 1), b01 = __ldg(pb), b23 = __ldg(pb + 1);
            const float2 a[4] = {make_float2(a01.x, a01.y), make_float2(a01.z, a01.w), make_float2(a23.x, a23.y),
                                 make_float2(a23.z, a23.w)};
            const float2 b[4] = {make_float2(b01.x, b01.y), make_float2(b01.z, b01.w), make_float2(b23.x, b23.y),
                                 make_float2(b23.z, b23.w)};
#pragma unroll
            for (int u = 0; u < 4; ++u)  // (cos, sin)(alpha + beta)
              cs[4 * h4 + u] = make_float2(fmaf(a[u].x, b[u].x, -(a[u].y * b[u].y)), fmaf(a[u].y, b[u].x, a[u].x * b[u].y));
          }
          // x chunk: column block 0, chunk pc;  y chunk: D = 128 -> column block 1, chunk pc;  D = 64 -> chunk pc + 4
          const int ycb = (D == 128) ? 1 : 0, ych = (D == 128) ? pc : pc + 4;
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            const int rr = hh * 64 + tok;
            uint4* px = reinterpret_cast<uint4*>(qt + rr * 128 + ((pc ^ (rr & 7)) << 4));
            uint4* py = reinterpret_cast<uint4*>(qt + ycb * L::kHalfBytes + rr * 128 + ((ych ^ (rr & 7)) << 4));
            const uint4 xv = *px, yv = *py;
            const uint32_t xw[4] = {xv.x, xv.y, xv.z, xv.w}, yw[4] = {yv.x, yv.y, yv.z, yv.w};
            uint32_t xo[4], yo[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const float x0 = __uint_as_float(xw[u] << 16), x1 = __uint_as_float(xw[u] & 0xFFFF0000u);
              const float y0 = __uint_as_float(yw[u] << 16), y1 = __uint_as_float(yw[u] & 0xFFFF0000u);
              const float2 c0 = cs[2 * u], c1 = cs[2 * u + 1];
              xo[u] = cvt_bf16x2(fmaf(x0, c0.x, -(y0 * c0.y)), fmaf(x1, c1.x, -(y1 * c1.y)));
              yo[u] = cvt_bf16x2(fmaf(y0, c0.x, x0 * c0.y), fmaf(y1, c1.x, x1 * c1.y));
            }
            *px = make_uint4(xo[0], xo[1], xo[2], xo[3]);
            *py = make_uint4(yo[0], yo[1], yo[2], yo[3]);
          }
        }
        fence_proxy_async();  // the rotated tile becomes visible to the tensor core's shared-memory reads
        __syncwarp();
        if (lane == 0) mbar_arrive(BAR(L::QROT + t));
      }
    };
    if constexpr (kRawQ) {
      if ((int)blockIdx.x < prm.n_items) rotate_item(decode_item(blockIdx.x, prm));
    }
    for (int it = blockIdx.x; it < prm.n_items; it += gridDim.x) {
      const Item im = decode_item(it, prm);
      if constexpr (kRawQ) {
        if (it + (int)gridDim.x < prm.n_items) rotate_item(decode_item(it + gridDim.x, prm));
      }
      for (int t = 0; t < im.nt; ++t) {
        mbar_wait(BAR(L::OFULL + t), o_cnt[t] & 1u);
        mbar_wait(BAR(L::LFULL + t), o_cnt[t] & 1u);
        ++o_cnt[t];
        tc_fence_after();
        float inv = s_invl[t * 128 + e * 32 + lane];
        const int head_in_group = (im.mt0 + t) * 2 + e / 2;
        const bool live = head_in_group < prm.G;
        const int grow = (im.b * prm.Hq + im.kv * prm.G + head_in_group) * prm.N + im.j * kChunk + (e % 2) * 32;
        const uint32_t o_addr = tmem + lane_base + (uint32_t)(256 + t * D);
        float w1 = 0.f;  // split mode: weight of the second partial result O_1 (0 when it saw no key tile)
        if constexpr (kSplit) {
          // merge the two partial softmax results of the item's single query tile (t == 0 here):
          // m = max(m0, m1), l = l0 2^(m0-m) + l1 2^(m1-m), O = (O_0 2^(m0-m) + O_1 2^(m1-m)) / l
          mbar_wait(BAR(L::OFULL + 1), o_cnt[1] & 1u);
          mbar_wait(BAR(L::LFULL + 1), o_cnt[1] & 1u);
          ++o_cnt[1];
          tc_fence_after();
          const int rowi = e * 32 + lane;
          const float l0 = inv, m0 = s_m[rowi], l1 = s_invl[128 + rowi], m1 = s_m[128 + rowi];
          const bool use1 = l1 > 0.f;
          const float m = use1 ? fmaxf(m0, m1) : m0;  // m0 is finite: tile 0 holds the diagonal key
          const float w0 = exp2f(m0 - m);
          w1 = use1 ? exp2f(m1 - m) : 0.f;
          const float l = l0 * w0 + l1 * w1;
          inv = w0 / l;
          w1 = w1 / l;
          if (lse != nullptr && live) {
            const size_t orow = ((size_t)im.b * prm.Hq + (size_t)(im.kv * prm.G + head_in_group)) * prm.N +
                                (size_t)im.j * kChunk + (size_t)(rowi % 64);
            lse[orow] = (m + log2f(l)) * 0.69314718055994530942f;
          }
        }
        // columns [c, c + 32) of the normalised output row into dst
        auto load_out = [&](int c, uint32_t* dst) {
          tmem_ld32(o_addr + c, dst);
          tmem_wait_ld();
#pragma unroll
          for (int u = 0; u < 32; ++u) dst[u] = __float_as_uint(__uint_as_float(dst[u]) * inv);
          if constexpr (kSplit) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              uint32_t o1[16];
              tmem_ld16(o_addr + D + c + 16 * h, o1);  // O_1 sits D columns after O_0
              tmem_wait_ld();
#pragma unroll
              for (int u = 0; u < 16; ++u)
                if (w1 != 0.f) dst[16 * h + u] = __float_as_uint(fmaf(__uint_as_float(o1[u]), w1, __uint_as_float(dst[16 * h + u])));
            }
          }
        };
        for (int c0 = 0; c0 < D; c0 += colw) {
          uint32_t w[32];
          if (prm.out_bf16) {
            uint32_t orr[32];
            load_out(c0, orr);
#pragma unroll
            for (int c = 0; c < 16; ++c) w[c] = cvt_bf16x2(__uint_as_float(orr[2 * c]), __uint_as_float(orr[2 * c + 1]));
            load_out(c0 + 32, orr);
#pragma unroll
            for (int c = 0; c < 16; ++c) w[16 + c] = cvt_bf16x2(__uint_as_float(orr[2 * c]), __uint_as_float(orr[2 * c + 1]));
          } else {
            load_out(c0, w);
          }
          if (live) {
            if (lane == 0) bulk_wait_read0();  // the previous store has finished reading the staging tile
            __syncwarp();
#pragma unroll
            for (int c = 0; c < 8; ++c)  // row `lane`, 16-byte chunk c at its 128B-swizzled position
              *reinterpret_cast<uint4*>(stage_p + lane * 128 + ((c ^ (lane & 7)) << 4)) =
                  make_uint4(w[4 * c], w[4 * c + 1], w[4 * c + 2], w[4 * c + 3]);
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) {
              tma_store_2d_hint(&tmO, stage, c0, grow, pol_o);
              bulk_commit();
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(BAR(L::OEMPTY + t));
          mbar_arrive(BAR(L::LEMPTY + t));
          if constexpr (kSplit) {
            mbar_arrive(BAR(L::OEMPTY + 1));
            mbar_arrive(BAR(L::LEMPTY + 1));
          }
        }
      }
    }
    if (lane == 0) bulk_wait0();
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsCtl));
    if (warp == kListWarp) {
      // ===================================== key-list builder ===================================================
      const int ppc = kChunk / 16, ppg = prm.gs / 16;
      int k = 0;
      for (int it = blockIdx.x; it < prm.n_items; it += gridDim.x, ++k) {
        const Item im = decode_item(it, prm);
        const int buf = k & 1;
        mbar_wait(BAR(L::LISTEMPTY + buf), ((uint32_t)(k >> 1) & 1u) ^ 1u);
        int* list = s_list + buf * prm.list_cap;
        const int j = im.j;
        const int n_sink = min(prm.F, j);
        const int loc_lo = max(max(0, j - prm.L_eff), n_sink);  // local chunks not already in the sink window
        const int n_loc = max(0, j - loc_lo);
        int n = 0;
        for (int i = lane; i < ppc; i += 32) list[i] = j * ppc + i;  // current chunk first
        n += ppc;
        for (int i = lane; i < n_sink * ppc; i += 32) list[n + i] = i;
        n += n_sink * ppc;
        // routed: closed earlier groups outside the sink/local windows (set union), compacted in list order so
        // that the summation order of the softmax is the same on every run
        if (group_idx != nullptr) {
          const int32_t* gi = group_idx + (((size_t)im.b * prm.Hkv + im.kv) * prm.n_b + j) * prm.Kg;
          for (int i0 = 0; i0 < prm.Kg; i0 += 32) {
            const int i = i0 + lane;
            const int g = (i < prm.Kg) ? __ldg(gi + i) : -1;
            bool keep = false;
            if (g >= 0) {
              const int c = (g * prm.gs) / kChunk;
              keep = (c < j) && !(c < n_sink) && !(c >= loc_lo);
            }
            const unsigned m = __ballot_sync(0xffffffffu, keep);
            if (keep) {
              const int slot = n + __popc(m & ((1u << lane) - 1u)) * ppg;
              for (int u = 0; u < ppg; ++u) list[slot + u] = g * ppg + u;
            }
            n += __popc(m) * ppg;
          }
        }
        for (int i = lane; i < n_loc * ppc; i += 32) list[n + i] = loc_lo * ppc + i;
        n += n_loc * ppc;
        __syncwarp();
        if (lane == 0) {
          s_np[buf] = n;
          mbar_arrive(BAR(L::LISTFULL + buf));
        }
      }
    } else if (warp == kLoadWarp) {
      // ===================================== TMA producer =======================================================
      const uint64_t pol_kv = policy_evict_last(), pol_q = policy_evict_first();
      uint32_t fill = 0;  // K/V tiles issued so far (both rings advance together)
      uint32_t qe_cnt[2] = {0, 0};  // Q tiles loaded per slot
      int k = 0;
      for (int it = blockIdx.x; it < prm.n_items; it += gridDim.x, ++k) {
        const Item im = decode_item(it, prm);
        const int buf = k & 1;
        mbar_wait(BAR(L::LISTFULL + buf), (uint32_t)(k >> 1) & 1u);
        const int n_pieces = s_np[buf];
        const int* list = s_list + buf * prm.list_cap;
        const int n_tiles = (n_pieces + kPPT - 1) / kPPT;
        const int kv_row0 = (im.b * prm.Hkv + im.kv) * prm.N;  // row of token 0 in the flattened [B*Hkv*N, D] K/V
        for (int i = 0; i < n_tiles; ++i, ++fill) {
          const int s = (int)(fill % L::kStages);
          const uint32_t ph = (fill / L::kStages) & 1u;
          const int np = min(kPPT, n_pieces - i * kPPT);
          const uint32_t bytes = (uint32_t)(np * 16 * D * 2);
          const int pc = lane / L::kHalves, cb = lane % L::kHalves;
          const bool active = lane < kPPT * L::kHalves && pc < np;
          const int row = active ? kv_row0 + list[i * kPPT + pc] * 16 : 0;
          const uint32_t off = (uint32_t)(s * L::kTileBytes + cb * L::kHalfBytes + pc * 16 * 128);
          mbar_wait(BAR(L::KEMPTY + s), ph ^ 1u);
          if (kDiag & 8) {
            if (lane == 0) mbar_arrive(BAR(L::KFULL + s));
          } else {
            if (lane == 0) mbar_expect_tx(BAR(L::KFULL + s), bytes);
            __syncwarp();
            if (active) tma_load_2d_hint(sbase + L::kK + off, &tmK, cb * 64, row, BAR(L::KFULL + s), pol_kv);
          }
          if (i == 0) {
            // Q tiles of this item: (tile t, head-in-tile hh, column block cb) -> 64 rows x 64 columns
            for (int t = 0; t < (kSplit ? 2 : im.nt); ++t) {  // split mode: the same Q tile in both slots
              mbar_wait(BAR(L::QEMPTY + t), (qe_cnt[t] & 1u) ^ 1u);
              ++qe_cnt[t];
              if (lane == 0) mbar_expect_tx(BAR(L::QFULL + t), (uint32_t)L::kTileBytes);
              __syncwarp();
              if (lane < 2 * L::kHalves) {
                const int qcb = lane % L::kHalves, hh = lane / L::kHalves;
                const int tq = kSplit ? 0 : t;
                int head_in_group = (im.mt0 + tq) * 2 + hh;
                if (head_in_group >= prm.G) head_in_group = (im.mt0 + tq) * 2;  // odd G: duplicate a live head, never stored
                const int qrow = (im.b * prm.Hq + im.kv * prm.G + head_in_group) * prm.N + im.j * kChunk;
                tma_load_2d_hint(sbase + L::kQ + t * L::kTileBytes + qcb * L::kHalfBytes + hh * 64 * 128, &tmQ, qcb * 64,
                                 qrow, BAR(L::QFULL + t), pol_q);
              }
            }
          }
          mbar_wait(BAR(L::VEMPTY + s), ph ^ 1u);
          if (kDiag & 8) {
            if (lane == 0) mbar_arrive(BAR(L::VFULL + s));
          } else {
            if (lane == 0) mbar_expect_tx(BAR(L::VFULL + s), bytes);
            __syncwarp();
            if (active) tma_load_2d_hint(sbase + L::kV + off, &tmV, cb * 64, row, BAR(L::VFULL + s), pol_kv);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(BAR(L::LISTEMPTY + buf));
      }
    } else if (warp == kMmaWarp) {
      // ===================================== MMA issuer ==========================================================
      // The whole warp runs the control flow convergently (so operands stay warp-uniform and ptxas needs no
      // per-lane broadcast loops); only the tcgen05 instructions themselves are predicated on one elected lane.
      const uint32_t ld = elect_one();
      const uint32_t tmem_u = uni(tmem);  // warp-uniform for ptxas: descriptors and addresses stay in uniform registers
      const uint32_t ldm = (kDiag & 2) ? 0u : ld;  // MMA issue predicate
      const uint32_t idesc_pv = umma_idesc(128, D, /*b_mn_major=*/true);
      const uint32_t idesc_qk_full = umma_idesc(128, kTileKeys, false);
      // descriptor high words are constant: SBO = 1024 B, version 1, SWIZZLE_128B
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
      constexpr uint32_t kLboK = (16u >> 4) << 16;                      // K-major operands (Q, K)
      constexpr uint32_t kLboV = ((uint32_t)L::kHalfBytes >> 4) << 16;  // MN-major V: next 64 columns
      auto issue_qk = [&](int t, int s, int nkeys) {
        const uint32_t idesc = nkeys == kTileKeys ? idesc_qk_full : umma_idesc(128, nkeys, false);
        const uint32_t qa = ((sbase + L::kQ + t * L::kTileBytes) & 0x3FFFFu) >> 4;
        const uint32_t ka = ((sbase + L::kK + s * L::kTileBytes) & 0x3FFFFu) >> 4;
        const uint32_t d = tmem_u + (uint32_t)(t * 128);
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t o = (uint32_t)((kk / 4) * L::kHalfBytes + (kk % 4) * 32) >> 4;
          umma_ss_e(d, make_desc(qa + o + kLboK, kDescHi), make_desc(ka + o + kLboK, kDescHi), idesc, kk > 0 ? 1u : 0u, ldm);
        }
      };
      auto issue_pv = [&](int t, int s, int kk0, int kk1, bool first) {
        const uint32_t va = ((sbase + L::kV + s * L::kTileBytes) & 0x3FFFFu) >> 4;
        const uint32_t d = tmem_u + (uint32_t)(256 + t * D);
        const uint32_t a = tmem_u + (uint32_t)(t * 128);
        // A: P_t columns [8kk, 8kk+8) (16 bf16 keys); B: V rows 16kk..16kk+15, MN-major
        if (kk1 - kk0 == kPPT / 2) {
#pragma unroll
          for (int u = 0; u < kPPT / 2; ++u) {
            const int kk = kk0 + u;
            umma_ts_e(d, a + (uint32_t)(kk * 8), make_desc(va + (uint32_t)(kk * 16 * 128 >> 4) + kLboV, kDescHi), idesc_pv,
                      (!first || kk > 0) ? 1u : 0u, ldm);
          }
        } else {
          for (int kk = kk0; kk < kk1; ++kk)
            umma_ts_e(d, a + (uint32_t)(kk * 8), make_desc(va + (uint32_t)(kk * 16 * 128 >> 4) + kLboV, kDescHi), idesc_pv,
                      (!first || kk > 0) ? 1u : 0u, ldm);
        }
      };
      if constexpr (kSplit) {
        // One query tile per item, two accumulators: virtual tile t (S_t, O_t, softmax warpgroup t) takes key tiles
        // u = t, t+2, ...; each has its own softmax -> P V -> Q K^T chain, so the two chains overlap on the tensor
        // pipe exactly like the two query tiles of the general case.  Key tile u of the item lives in stage
        // (base + u) % kStages and is used by one virtual tile only.
        uint32_t base = 0, q_cnt[2] = {0, 0}, p_cnt[2] = {0, 0}, oe_cnt[2] = {0, 0};
        // first Q K^T of virtual tile t for an item of np pieces whose key tile 0 is global tile b0
        auto first_qk = [&](int t, int np, uint32_t b0) {
          const int nt_ = (np + kPPT - 1) / kPPT;
          mbar_wait(BAR((kRawQ ? L::QROT : L::QFULL) + t), q_cnt[t] & 1u);
          ++q_cnt[t];
          if (t < nt_) {
            const int ks = (int)((b0 + (uint32_t)t) % L::kStages);
            mbar_wait(BAR(L::KFULL + ks), ((b0 + (uint32_t)t) / L::kStages) & 1u);
            tc_fence_after();
            issue_qk(t, ks, min(kPPT, np - t * kPPT) * 16);
            umma_commit_e(BAR(L::SFULL + t), ld);
            umma_commit_e(BAR(L::KEMPTY + ks), ld);
            if (t + 2 >= nt_) umma_commit_e(BAR(L::QEMPTY + t), ld);
          } else if (ld) {
            mbar_arrive(BAR(L::QEMPTY + t));  // this half has no key tile: its Q slot is free at once
          }
        };
        bool pre[2] = {false, false};  // the next item's first Q K^T of tile t went out behind this item's last P V
        int k = 0;
        for (int it = blockIdx.x; it < prm.n_items; it += gridDim.x, ++k) {
          const int buf = k & 1;
          const bool has_next = it + (int)gridDim.x < prm.n_items;
          mbar_wait(BAR(L::LISTFULL + buf), (uint32_t)(k >> 1) & 1u);
          const int n_pieces = uni(s_np[buf]);
          const int n_tiles = (n_pieces + kPPT - 1) / kPPT;
          auto nkeys_of = [&](int u) { return min(kPPT, n_pieces - u * kPPT) * 16; };
          auto st_of = [&](int u) { return (int)((base + (uint32_t)u) % L::kStages); };
          auto ph_of = [&](int u) { return ((base + (uint32_t)u) / L::kStages) & 1u; };
          for (int t = 0; t < 2; ++t) {
            if (!pre[t]) first_qk(t, n_pieces, base);
            pre[t] = false;
          }
          for (int u = 0; u < n_tiles; ++u) {
            const int t = u & 1, vs = st_of(u), nkeys = nkeys_of(u);
            mbar_wait(BAR(L::PFULL + t), p_cnt[t] & 1u);  // keys 0..63 of P_t
            if (u < 2) {
              mbar_wait(BAR(L::OEMPTY + t), (oe_cnt[t] & 1u) ^ 1u);  // the epilogue has drained the previous item's O_t
              ++oe_cnt[t];
            }
            mbar_wait(BAR(L::VFULL + vs), ph_of(u));
            tc_fence_after();
            issue_pv(t, vs, 0, min(nkeys / 16, kPPT / 2), u < 2);
            mbar_wait(BAR(L::PFULLB + t), p_cnt[t] & 1u);  // keys 64..127
            ++p_cnt[t];
            tc_fence_after();
            issue_pv(t, vs, kPPT / 2, nkeys / 16, false);
            umma_commit_e(BAR(L::VEMPTY + vs), ld);
            if (u + 2 < n_tiles) {
              const int ks = st_of(u + 2);
              mbar_wait(BAR(L::KFULL + ks), ph_of(u + 2));
              tc_fence_after();
              issue_qk(t, ks, nkeys_of(u + 2));
              umma_commit_e(BAR(L::SFULL + t), ld);
              umma_commit_e(BAR(L::KEMPTY + ks), ld);
              if (u + 4 >= n_tiles) umma_commit_e(BAR(L::QEMPTY + t), ld);
            } else {
              umma_commit_e(BAR(L::OFULL + t), ld);
              if (has_next) {
                // S_t is free once this P V has run: queue the next item's first Q K^T of this tile right behind it
                mbar_wait(BAR(L::LISTFULL + (buf ^ 1)), (uint32_t)((k + 1) >> 1) & 1u);
                first_qk(t, uni(s_np[buf ^ 1]), base + (uint32_t)n_tiles);
                pre[t] = true;
              }
            }
          }
          if (n_tiles < 2) {
            // the second half saw no key tile (block 0 with a 64-key list): hand its untouched O_1 over anyway, the
            // epilogue gives it weight 0
            mbar_wait(BAR(L::OEMPTY + 1), (oe_cnt[1] & 1u) ^ 1u);
            ++oe_cnt[1];
            if (ld) mbar_arrive(BAR(L::OFULL + 1));
          }
          base += (uint32_t)n_tiles;
          __syncwarp();
          if (lane == 0) mbar_arrive(BAR(L::LISTEMPTY + buf));
        }
      }
      // General case (two query tiles per item).  The issuer warp is a serial instruction stream, and at 64 cycles
      // per MMA it -- not the tensor pipe -- sets the pace as soon as it spends more than that per instruction
      // (descriptor words moved from vector to uniform registers, ~100 cycles per barrier wait): measured 3,300
      // cycles per key-tile step against 2,048 of MMA work.  So the key-tile step is instantiated once per ring
      // stage: the tile and stage indices are compile-time constants and every descriptor is a constant offset from
      // the (uniform) shared-memory base.
      uint32_t step = 0;  // K/V tiles consumed so far: tile `step` lives in stage step % kStages
      int k = 0;
      int it = kSplit ? prm.n_items : blockIdx.x;  // split mode is handled above
      int n_pieces = 0, nt = 0;
      uint32_t q_cnt[2] = {0, 0}, p_cnt[2] = {0, 0}, oe_cnt[2] = {0, 0};
      const uint32_t sb4 = (sbase & 0x3FFFFu) >> 4;  // tile bases are 1024-byte aligned: offsets add without carry
      auto qk = [&](auto T, auto S, int nkeys) {
        constexpr int t = decltype(T)::value, st = decltype(S)::value;
        const uint32_t idesc = nkeys == kTileKeys ? idesc_qk_full : umma_idesc(128, nkeys, false);
        const uint32_t d = tmem_u + (uint32_t)(t * 128);
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          constexpr uint32_t kZero = 0;
          const uint32_t o = (uint32_t)((kk / 4) * L::kHalfBytes + (kk % 4) * 32) >> 4;
          const uint32_t qo = ((uint32_t)(L::kQ + t * L::kTileBytes) >> 4) + o + kLboK + kZero;
          const uint32_t ko = ((uint32_t)(L::kK + st * L::kTileBytes) >> 4) + o + kLboK;
          umma_ss_e(d, make_desc(sb4 + qo, kDescHi), make_desc(sb4 + ko, kDescHi), idesc, kk > 0 ? 1u : 0u, ldm);
        }
      };
      auto pv = [&](auto T, auto S, int kk0, int kk1, bool first) {
        constexpr int t = decltype(T)::value, st = decltype(S)::value;
        const uint32_t d = tmem_u + (uint32_t)(256 + t * D);
        const uint32_t a = tmem_u + (uint32_t)(t * 128);
        // A: P_t columns [8kk, 8kk+8) (16 bf16 keys); B: V rows 16kk..16kk+15, MN-major
        auto one = [&](int kk, uint32_t acc) {
          const uint32_t vo = ((uint32_t)(L::kV + st * L::kTileBytes + kk * 16 * 128) >> 4) + kLboV;
          umma_ts_e(d, a + (uint32_t)(kk * 8), make_desc(sb4 + vo, kDescHi), idesc_pv, acc, ldm);
        };
        if (kk1 - kk0 == kPPT / 2) {  // a whole half tile: no per-instruction branches
          if (kk0 == 0) {
            one(0, first ? 0u : 1u);
            one(1, 1u);
            one(2, 1u);
            one(3, 1u);
          } else {
            one(4, 1u);
            one(5, 1u);
            one(6, 1u);
            one(7, 1u);
          }
        } else {
#pragma unroll
          for (int kk = 0; kk < kPPT; ++kk)
            if (kk >= kk0 && kk < kk1) one(kk, (!first || kk > 0) ? 1u : 0u);
        }
      };
      if (it < prm.n_items) {
        mbar_wait(BAR(L::LISTFULL + 0), 0);
        n_pieces = uni(s_np[0]);
        nt = decode_item(it, prm).nt;
        // first Q K^T of the first item
        mbar_wait(BAR(L::KFULL + 0), 0);
        auto first_qk = [&](auto T) {
          constexpr int t = decltype(T)::value;
          if (t < nt) {
            mbar_wait(BAR((kRawQ ? L::QROT : L::QFULL) + t), 0);
            ++q_cnt[t];
            tc_fence_after();
            qk(T, std::integral_constant<int, 0>{}, min(kPPT, n_pieces) * 16);
            umma_commit_e(BAR(L::SFULL + t), ld);
            if (n_pieces <= kPPT) umma_commit_e(BAR(L::QEMPTY + t), ld);
          }
        };
        first_qk(std::integral_constant<int, 0>{});
        first_qk(std::integral_constant<int, 1>{});
        umma_commit_e(BAR(L::KEMPTY + 0), ld);
      }
      for (; it < prm.n_items; it += gridDim.x, ++k) {
        const int buf = k & 1;
        const int n_tiles = (n_pieces + kPPT - 1) / kPPT;
        const int it_next = it + gridDim.x;
        const bool has_next = it_next < prm.n_items;
        int n_pieces_next = 0, nt_next = 0;
        for (int i = 0; i < n_tiles; ++i, ++step) {
          const bool last = (i + 1 == n_tiles);
          const bool more = !last || has_next;  // another Q K^T follows this tile's P V
          int nkeys_next = 0, n_tiles_after = 0;
          if (!last) {
            nkeys_next = min(kPPT, n_pieces - (i + 1) * kPPT) * 16;
            n_tiles_after = n_tiles - (i + 2);
          } else if (has_next) {
            mbar_wait(BAR(L::LISTFULL + (buf ^ 1)), (uint32_t)((k + 1) >> 1) & 1u);
            n_pieces_next = uni(s_np[buf ^ 1]);
            nt_next = decode_item(it_next, prm).nt;
            nkeys_next = min(kPPT, n_pieces_next) * 16;
            n_tiles_after = (n_pieces_next + kPPT - 1) / kPPT - 1;
          }
          const int nkeys = min(kPPT, n_pieces - i * kPPT) * 16;
          const int nt_qk = last ? nt_next : nt;
          const uint32_t v_ph = (step / L::kStages) & 1u, k_ph = ((step + 1) / L::kStages) & 1u;
          // one key-tile step with the V tile in stage VS and the next K tile in stage KS
          auto tile_step = [&](auto VS) {
            constexpr int vs = decltype(VS)::value, ks = (vs + 1) % L::kStages;
            using KS = std::integral_constant<int, ks>;
            mbar_wait(BAR(L::VFULL + vs), v_ph);
            if (more) mbar_wait(BAR(L::KFULL + ks), k_ph);
            auto one = [&](auto T) {
              constexpr int t = decltype(T)::value;
              const bool tron = blockIdx.x == 0 && k >= 8 && k < 10 && i < 8;
              const int trs = 1024 + (((k - 8) * 8 + i) * 2 + t) * 8;
              (void)tron;
              (void)trs;
              if (t < nt) {
                mbar_wait(BAR(L::PFULL + t), p_cnt[t] & 1u);  // keys 0..63 of P_t
                HGA_TRM(trs + 0);
                if (i == 0) {
                  // the epilogue has drained the previous item's O_t
                  mbar_wait(BAR(L::OEMPTY + t), (oe_cnt[t] & 1u) ^ 1u);
                  ++oe_cnt[t];
                }
                tc_fence_after();
                pv(T, VS, 0, min(nkeys / 16, kPPT / 2), i == 0);
                HGA_TRM(trs + 1);
                mbar_wait(BAR(L::PFULLB + t), p_cnt[t] & 1u);  // keys 64..127
                HGA_TRM(trs + 2);
                ++p_cnt[t];
                tc_fence_after();
                pv(T, VS, kPPT / 2, nkeys / 16, false);
                if (last) umma_commit_e(BAR(L::OFULL + t), ld);
              }
              if (more && t < nt_qk) {
                if (last) {
                  mbar_wait(BAR((kRawQ ? L::QROT : L::QFULL) + t), q_cnt[t] & 1u);
                  ++q_cnt[t];
                  tc_fence_after();
                }
                qk(T, KS{}, nkeys_next);
                umma_commit_e(BAR(L::SFULL + t), ld);
                if (n_tiles_after == 0) umma_commit_e(BAR(L::QEMPTY + t), ld);  // that was the item's last Q K^T
              }
              HGA_TRM(trs + 3);
            };
            one(std::integral_constant<int, 0>{});
            one(std::integral_constant<int, 1>{});
            umma_commit_e(BAR(L::VEMPTY + vs), ld);
            if (more) umma_commit_e(BAR(L::KEMPTY + ks), ld);
          };
          const uint32_t vsi = step % L::kStages;
          if constexpr (L::kStages == 2) {
            if (vsi == 0) tile_step(std::integral_constant<int, 0>{});
            else tile_step(std::integral_constant<int, 1>{});
          } else {
            if (vsi == 0) tile_step(std::integral_constant<int, 0>{});
            else if (vsi == 1) tile_step(std::integral_constant<int, 1>{});
            else if (vsi == 2) tile_step(std::integral_constant<int, 2>{});
            else tile_step(std::integral_constant<int, 3>{});
          }
        }
        if (lane == 0) mbar_arrive(BAR(L::LISTEMPTY + buf));
        n_pieces = n_pieces_next;
        nt = nt_next;
      }
      __syncwarp();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kMmaWarp) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

// rope_a / rope_b non-null: q holds the UN-rotated queries and the kernel applies RoPE itself (kRawQ)
template <int D>
hga_status launch_tc2_t(const Derived& d, const void* q, const void* k, const void* v, const int32_t* gi, void* out,
                        float* lse, const float2* rope_a, const float2* rope_b, cudaStream_t s) {
  using L = Smem2<D>;
  Tc2Params prm;
  prm.B = d.B; prm.Hq = d.Hq; prm.Hkv = d.Hkv; prm.N = d.N; prm.n_b = d.n_b; prm.G = d.G;
  prm.jb = d.jb; prm.nj = d.nj;
  prm.F = d.F; prm.L_eff = d.L_eff; prm.gs = d.gs; prm.Kg = d.Kg;
  prm.n_mt = (d.G + 1) / 2;
  prm.ctas_per_unit = (prm.n_mt + 1) / 2;
  prm.split = prm.n_mt == 1 ? 1 : 0;
  prm.list_cap = max_key_pieces(d.F, d.L_eff, d.gs, d.Kg);
  prm.scale_log2 = d.scale * 1.4426950408889634f;
  prm.out_bf16 = d.bf16_out ? 1 : 0;
  prm.rope_a = rope_a;
  prm.rope_b = rope_b;
  const long long n_items = (long long)d.B * d.Hkv * d.nj * prm.ctas_per_unit;
  const size_t smem = (size_t)L::kList + 2 * sizeof(int) * (size_t)prm.list_cap;
  if (smem > 227 * 1024 || n_items >= (1ll << 31)) return HGA_ERR_UNSUPPORTED;
  if ((uint64_t)d.B * d.Hq * d.N >= (1ull << 31)) return HGA_ERR_UNSUPPORTED;
  prm.n_items = (int)n_items;
  CUtensorMap tmQ, tmK, tmV, tmO;
  const uint64_t q_rows = (uint64_t)d.B * d.Hq * d.N, kv_rows = (uint64_t)d.B * d.Hkv * d.N;
  bool ok = make_map_2d(&tmQ, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, q, q_rows, D, 64, 64) &&
            make_map_2d(&tmK, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, k, kv_rows, D, 64, 16) &&
            make_map_2d(&tmV, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, v, kv_rows, D, 64, 16);
  ok = ok && (d.bf16_out ? make_map_2d(&tmO, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, out, q_rows, D, 64, 32)
                         : make_map_2d(&tmO, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, out, q_rows, D, 32, 32));
  if (!ok) return HGA_ERR_CUDA;
  const int n_sm = current_sm_count();
  if (n_sm <= 0) return HGA_ERR_CUDA;
  const bool raw = rope_a != nullptr && rope_b != nullptr;
  auto kern = prm.split ? (raw ? attend_tc2_kernel<D, true, true, true> : attend_tc2_kernel<D, true, true, false>)
              : d.G % 2 ? (raw ? attend_tc2_kernel<D, false, true, true> : attend_tc2_kernel<D, false, true, false>)
                        : (raw ? attend_tc2_kernel<D, false, false, true> : attend_tc2_kernel<D, false, false, false>);
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int grid = (int)(n_items < n_sm ? n_items : n_sm);
  kern<<<grid, kThreads, smem, s>>>(tmQ, tmK, tmV, tmO, gi, lse, prm);
  return launch_status();
}

}  // namespace

#ifdef HGA_S4_TRACE
extern "C" __attribute__((visibility("default"))) int hga_debug_trace(long long* host_out) {
  return (int)cudaMemcpyFromSymbol(host_out, g_trace, sizeof(long long) * 4096);
}
#endif

// Returns HGA_ERR_UNSUPPORTED when the key list does not fit beside the tiles (the caller falls back to the
// one-item-per-CTA kernel).
hga_status launch_attend_tc2(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                             void* out, float* lse, cudaStream_t s) {
  if (!d.bf16_io) return HGA_ERR_UNSUPPORTED;
  return d.D == 128 ? launch_tc2_t<128>(d, q, k, v, group_idx, out, lse, nullptr, nullptr, s)
                    : launch_tc2_t<64>(d, q, k, v, group_idx, out, lse, nullptr, nullptr, s);
}

// N2: the same kernel on UN-rotated queries; RoPE is applied to every Q tile inside the kernel from the two position
// tables of launch_rope_tables (rope_a: [n_b][D/2], rope_b: [64][D/2]), so Q_rot never goes through HBM.
hga_status launch_attend_tc2_rawq(const Derived& d, const void* q_raw, const void* k, const void* v, const int32_t* group_idx,
                                  void* out, float* lse, const float2* rope_a, const float2* rope_b, cudaStream_t s) {
  if (!d.bf16_io || !rope_a || !rope_b) return HGA_ERR_UNSUPPORTED;
  return d.D == 128 ? launch_tc2_t<128>(d, q_raw, k, v, group_idx, out, lse, rope_a, rope_b, s)
                    : launch_tc2_t<64>(d, q_raw, k, v, group_idx, out, lse, rope_a, rope_b, s);
}

}  // namespace hga
