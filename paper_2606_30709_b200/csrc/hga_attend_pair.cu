// S4 for whole GQA groups of 8 query heads at head_dim 128 (the Qwen3-30B-A3B shape of c4 / c5 / p5): one CTA PAIR
// (a 2-CTA cluster on one TPC) per (batch, kv head, query block j) unit, tcgen05.mma.cta_group::2.
// (Eq. (1) PAPER.md:56 over the union set.)
//
// Why a pair: the four 128-row query tiles of a unit (8 heads x 64 tokens) all read the SAME gathered K/V.  With one
// CTA per two tiles (attend_tc2_kernel) every K/V tile travels L2 -> shared memory twice and the kernel's memory
// skeleton alone (TMA gathers + barriers, no MMA, no softmax) takes 0.60 ms at c5 -- the L2 -> SM fabric, not the
// tensor pipe, is the floor.  Here each CTA of the pair holds two query tiles and HALF of every K/V tile:
//   Q K^T : M = 256 (rows 0..127 = this CTA's tile, 128..255 = the peer's), N = keys of the tile, split by N --
//           the leader CTA supplies the first half of the keys, the peer the second half;
//   P V   : M = 256, N = D = 128 split by N -- each CTA supplies 64 of the 128 V columns for all keys.
// So L2 -> SM traffic and the shared-memory reads of the B operand halve, and the freed shared memory doubles the
// K/V ring (4 stages each).  One thread of the leader CTA issues every MMA of the pair; completions are multicast
// to the barriers of both CTAs, and the peer's softmax / epilogue / producer warps signal the leader's barriers
// through shared::cluster addresses.
//
//   warps 0-3 / 4-7  softmax warpgroups (query tile slot 0 / 1 of this CTA), one thread per query row
//   warps 8-11       epilogue: O_u / l -> swizzled staging tile -> TMA store
//   warp 12          tcgen05.mma issuer (leader CTA only)
//   warp 13          TMA producer: this CTA's half of the K and V pieces, this CTA's two Q tiles
//   warp 14          key-list builder (each CTA builds the unit's list for itself)
//
// CTA r, slot u holds query tile 2r + u = heads (4r + 2u, 4r + 2u + 1) of the group.  TMEM map per CTA (512
// columns): S_u at 128u (P_u overlays its first 64 columns), O_u at 256 + 128u.  Key order inside a unit: current
// chunk first (the causal mask lives in columns 0..63 of tile 0), sink chunks, routed groups, local chunks; only the
// last 128-key tile can be partial: with np valid 16-key pieces the Q K^T runs at N = 32*ceil(np/2) (the leader
// holds the first ceil(np/2) pieces, the peer the rest) and the softmax masks the columns >= 16 np.
#include <cuda.h>
#include <math_constants.h>

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
constexpr int kD = 128;

struct PairParams {
  int B, Hq, Hkv, N, n_b, G;
  int jb, nj;  // query blocks [jb, jb + nj) of every (batch, kv head) are processed
  int F, L_eff, gs, Kg;
  int list_cap;  // pieces per list buffer
  int n_items;   // units
  float scale_log2;
  int out_bf16;
};

struct SmemP {
  static constexpr int kQHalf = 128 * 128;        // 128 rows x 128 B
  static constexpr int kQTile = 2 * kQHalf;       // 32 KB
  static constexpr int kKHalf = 64 * 128;         // this CTA's 64 keys x 128 B
  static constexpr int kKTile = 2 * kKHalf;       // 16 KB
  static constexpr int kVTile = kTileKeys * 128;  // 128 keys x this CTA's 64 columns = 16 KB
  static constexpr int kStages = 4;
  static constexpr int kQ = 0;
  static constexpr int kK = kQ + 2 * kQTile;
  static constexpr int kV = kK + kStages * kKTile;
  static constexpr int kStage = kV + kStages * kVTile;  // epilogue staging: 4 warps x 4 KB
  static constexpr int kBar = kStage + 4 * 4096;
  static constexpr int QFULL = 0, QEMPTY = 2, SFULL = 4, PFULL = 6, OFULL = 8, OEMPTY = 10, LFULL = 12, LEMPTY = 14,
                       LISTFULL = 16, LISTEMPTY = 18, PFULLB = 20, KFULL = 22, KEMPTY = KFULL + kStages,
                       VFULL = KEMPTY + kStages, VEMPTY = VFULL + kStages, kNumBars = VEMPTY + kStages;
  static constexpr int kMisc = kBar + 8 * kNumBars;  // tmem base (4 B), n_pieces[2]
  static constexpr int kInvL = kMisc + 16;           // 2 slots x 128 rows fp32: 1/l
  static constexpr int kList = kInvL + 2 * 128 * 4;  // 2 x list_cap ints
};

struct Unit {
  int b, kv, j;
};

__device__ __forceinline__ Unit decode_unit(int it, const PairParams& prm) {
  // (batch, kv head) outermost so one head's K/V stays L2-resident while its Q streams through; j descending
  // inside a head (longest lists first, the short early blocks fill the tail)
  Unit r;
  const int bk = it / prm.nj;
  r.j = prm.jb + prm.nj - 1 - it % prm.nj;
  r.kv = bk % prm.Hkv;
  r.b = bk / prm.Hkv;
  return r;
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
attend_pair_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                   const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmO,
                   const int32_t* __restrict__ group_idx, float* __restrict__ lse, const PairParams prm) {
  using L = SmemP;
  constexpr int D = kD;
  extern __shared__ __align__(1024) unsigned char smem[];
  const uint32_t sbase = smem_u32(smem);
  auto BAR = [&](int i) { return sbase + (uint32_t)L::kBar + 8u * (uint32_t)i; };
  volatile uint32_t* tmem_base_p = reinterpret_cast<volatile uint32_t*>(smem + L::kMisc);
  volatile int* s_np = reinterpret_cast<volatile int*>(smem + L::kMisc + 4);  // [2]
  float* s_invl = reinterpret_cast<float*>(smem + L::kInvL);                  // [2][128]
  int* s_list = reinterpret_cast<int*>(smem + L::kList);                      // [2][list_cap]

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const uint32_t rank = cluster_ctarank();  // 0 = leader (issues the MMAs, owns the cross-CTA barriers)
  const int pair = blockIdx.x / 2, n_pairs = gridDim.x / 2;
  auto LBAR = [&](int i) { return mapa(BAR(i), 0); };  // the leader's barrier i, as a shared::cluster address

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();  // the 128B-swizzled tiles need a 1024-byte aligned base
    for (int u = 0; u < 2; ++u) {
      mbar_init(BAR(L::QFULL + u), 2);   // both producers (arrive.expect_tx); leader's copy is the live one
      mbar_init(BAR(L::QEMPTY + u), 1);  // multicast commit
      mbar_init(BAR(L::SFULL + u), 1);   // multicast commit
      mbar_init(BAR(L::PFULL + u), 8);   // 4 softmax warps of each CTA; leader's copy
      mbar_init(BAR(L::PFULLB + u), 8);
      mbar_init(BAR(L::OFULL + u), 1);   // multicast commit
      mbar_init(BAR(L::OEMPTY + u), 8);  // 4 epilogue warps of each CTA; leader's copy
      mbar_init(BAR(L::LFULL + u), 4);
      mbar_init(BAR(L::LEMPTY + u), 4);
      mbar_init(BAR(L::LISTFULL + u), 1);
      mbar_init(BAR(L::LISTEMPTY + u), rank == 0 ? 10 : 9);  // producer + 8 softmax warps (+ the leader's MMA warp)
    }
    for (int s = 0; s < L::kStages; ++s) {
      mbar_init(BAR(L::KFULL + s), 2);  // both producers; leader's copy
      mbar_init(BAR(L::KEMPTY + s), 1);
      mbar_init(BAR(L::VFULL + s), 2);
      mbar_init(BAR(L::VEMPTY + s), 1);
    }
    fence_barrier_init();
    fence_proxy_async();
  }
  if (warp == kMmaWarp) tmem_alloc2(sbase + L::kMisc, 512);
  if (warp == kLoadWarp && lane == 0) {
    prefetch_tmap(&tmQ);
    prefetch_tmap(&tmK);
    prefetch_tmap(&tmV);
  }
  if (warp == kEpiWarp0 && lane == 0) prefetch_tmap(&tmO);
  tc_fence_before();
  cluster_sync_all();  // barrier inits and the TMEM allocation of both CTAs are visible to the pair
  tc_fence_after();
  const uint32_t tmem = *tmem_base_p;

  if (warp < 8) {
    // ===================================== softmax warpgroups ===================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsSoftmax));
    const int t = warp / 4;                  // query tile slot of this warpgroup
    const int row = (warp % 4) * 32 + lane;  // row of the 128-row tile == TMEM lane
    const int r64 = row % 64;
    const uint32_t lane_base = (uint32_t)((warp % 4) * 32) << 16;
    const uint32_t s_addr = tmem + lane_base + (uint32_t)(t * 128);
    const uint32_t o_addr = tmem + lane_base + (uint32_t)(256 + t * D);
    const float sl2 = prm.scale_log2;
    const uint32_t pfull = LBAR(L::PFULL + t), pfullb = LBAR(L::PFULLB + t);
    uint32_t s_cnt = 0;   // S_FULL completions consumed
    uint32_t n_done = 0;  // units this warpgroup has processed
    int k = 0;
    for (int it = pair; it < prm.n_items; it += n_pairs, ++k) {
      const Unit im = decode_unit(it, prm);
      const int buf = k & 1;
      mbar_wait(BAR(L::LISTFULL + buf), (uint32_t)(k >> 1) & 1u);
      const int n_pieces = s_np[buf];
      __syncwarp();
      if (lane == 0) mbar_arrive(BAR(L::LISTEMPTY + buf));
      const int n_tiles = (n_pieces + kPPT - 1) / kPPT;
      float m_run = -CUDART_INF_F;  // running reference max, raw logit units
      float l_run = 0.f;
      for (int i = 0; i < n_tiles; ++i) {
        const int nk = min(kPPT, n_pieces - i * kPPT) * 16;  // valid key columns of this tile
        mbar_wait(BAR(L::SFULL + t), s_cnt & 1u);
        ++s_cnt;
        if (kDiag & 1) {
          __syncwarp();
          if (lane == 0) {
            mbar_arrive_cluster(pfull);
            mbar_arrive_cluster(pfullb);
          }
          continue;
        }
        tc_fence_after();
        softmax_tile<D>(
            s_addr, o_addr, i == 0, r64, nk, i != 0, sl2, m_run, l_run,
            [&] {
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(pfull);
            },
            [&] {
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(pfullb);
            });
      }
      // ---- unit done: hand 1/l to the epilogue warpgroup, write LSE ----------------------------------------------
      mbar_wait(BAR(L::LEMPTY + t), (n_done & 1u) ^ 1u);
      ++n_done;
      s_invl[t * 128 + row] = 1.f / l_run;
      const int head_in_group = ((int)rank * 2 + t) * 2 + row / 64;
      if (lse != nullptr) {
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
    uint32_t o_cnt[2] = {0, 0};               // units drained per slot
    const uint64_t pol_o = policy_evict_first();
    for (int it = pair; it < prm.n_items; it += n_pairs) {
      const Unit im = decode_unit(it, prm);
      for (int t = 0; t < 2; ++t) {
        mbar_wait(BAR(L::OFULL + t), o_cnt[t] & 1u);
        mbar_wait(BAR(L::LFULL + t), o_cnt[t] & 1u);
        ++o_cnt[t];
        tc_fence_after();
        const float inv = s_invl[t * 128 + e * 32 + lane];
        const int head_in_group = ((int)rank * 2 + t) * 2 + e / 2;
        const int grow = (im.b * prm.Hq + im.kv * prm.G + head_in_group) * prm.N + im.j * kChunk + (e % 2) * 32;
        const uint32_t o_addr = tmem + lane_base + (uint32_t)(256 + t * D);
        auto load_out = [&](int c, uint32_t* dst) {  // columns [c, c + 32) of the normalised output row
          tmem_ld32(o_addr + c, dst);
          tmem_wait_ld();
#pragma unroll
          for (int u = 0; u < 32; ++u) dst[u] = __float_as_uint(__uint_as_float(dst[u]) * inv);
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
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive_cluster(LBAR(L::OEMPTY + t));  // the leader's MMA warp may overwrite O_t of both CTAs
          mbar_arrive(BAR(L::LEMPTY + t));
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
      for (int it = pair; it < prm.n_items; it += n_pairs, ++k) {
        const Unit im = decode_unit(it, prm);
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
      // K tile: this CTA's half of the pieces (leader: the first ceil(np/2), peer: the rest), both 64-column blocks;
      // V tile: every piece, this CTA's 64-column block.  Full barriers live in the leader CTA.
      const uint64_t pol_kv = policy_evict_last(), pol_q = policy_evict_first();
      uint32_t fill = 0;            // K/V tiles issued so far (both rings advance together)
      uint32_t qe_cnt[2] = {0, 0};  // Q tiles loaded per slot
      int k = 0;
      for (int it = pair; it < prm.n_items; it += n_pairs, ++k) {
        const Unit im = decode_unit(it, prm);
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
          const int nph = (np + 1) / 2;
          const int k_first = rank == 0 ? 0 : nph, k_cnt = rank == 0 ? nph : np - nph;
          // ---- K ----
          {
            const int pc = lane / 2, cb = lane % 2;
            const bool active = lane < 2 * k_cnt;
            const int row = active ? kv_row0 + list[i * kPPT + k_first + pc] * 16 : 0;
            const uint32_t off = (uint32_t)(s * L::kKTile + cb * L::kKHalf + pc * 16 * 128);
            const uint32_t full = LBAR(L::KFULL + s);
            mbar_wait(BAR(L::KEMPTY + s), ph ^ 1u);
            if (kDiag & 8) {
              if (lane == 0) mbar_arrive_cluster(full);
            } else {
              if (lane == 0) {
                if (k_cnt > 0) mbar_expect_tx_cluster(full, (uint32_t)(k_cnt * 16 * D * 2));
                else mbar_arrive_cluster(full);
              }
              __syncwarp();
              if (active) tma_load_2d_pair(sbase + L::kK + off, &tmK, cb * 64, row, full, pol_kv);
            }
          }
          if (i == 0) {
            // this CTA's two Q tiles: (slot u, head-in-tile hh, column block qcb) -> 64 rows x 64 columns
            for (int u = 0; u < 2; ++u) {
              mbar_wait(BAR(L::QEMPTY + u), (qe_cnt[u] & 1u) ^ 1u);
              ++qe_cnt[u];
              const uint32_t full = LBAR(L::QFULL + u);
              if (lane == 0) mbar_expect_tx_cluster(full, (uint32_t)L::kQTile);
              __syncwarp();
              if (lane < 4) {
                const int qcb = lane % 2, hh = lane / 2;
                const int head_in_group = ((int)rank * 2 + u) * 2 + hh;
                const int qrow = (im.b * prm.Hq + im.kv * prm.G + head_in_group) * prm.N + im.j * kChunk;
                tma_load_2d_pair(sbase + L::kQ + u * L::kQTile + qcb * L::kQHalf + hh * 64 * 128, &tmQ, qcb * 64, qrow, full,
                                 pol_q);
              }
            }
          }
          // ---- V ----
          {
            const bool active = lane < np;
            const int row = active ? kv_row0 + list[i * kPPT + lane] * 16 : 0;
            const uint32_t off = (uint32_t)(s * L::kVTile + lane * 16 * 128);
            const uint32_t full = LBAR(L::VFULL + s);
            mbar_wait(BAR(L::VEMPTY + s), ph ^ 1u);
            if (kDiag & 8) {
              if (lane == 0) mbar_arrive_cluster(full);
            } else {
              if (lane == 0) mbar_expect_tx_cluster(full, (uint32_t)(np * 16 * 64 * 2));
              __syncwarp();
              if (active) tma_load_2d_pair(sbase + L::kV + off, &tmV, (int)rank * 64, row, full, pol_kv);
            }
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(BAR(L::LISTEMPTY + buf));
      }
    } else if (warp == kMmaWarp && rank == 0) {
      // ===================================== MMA issuer (leader CTA) ==============================================
      // The whole warp runs the control flow convergently (operands stay warp-uniform); only the tcgen05
      // instructions themselves are predicated on one elected lane.
      const uint32_t ld = elect_one();
      const uint32_t tmem_u = uni(tmem);  // warp-uniform for ptxas: descriptors and addresses stay in uniform registers
      const uint32_t ldm = (kDiag & 2) ? 0u : ld;  // MMA issue predicate
      const uint32_t idesc_pv = umma_idesc(256, D, /*b_mn_major=*/true);
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);  // SBO = 1024 B, version 1, SWIZZLE_128B
      constexpr uint32_t kLbo = (16u >> 4) << 16;
      uint32_t q_cnt[2] = {0, 0}, p_cnt[2] = {0, 0}, oe_cnt[2] = {0, 0};
      auto issue_qk = [&](int u, int s, int np) {
        const uint32_t idesc = umma_idesc(256, 32 * ((np + 1) / 2), false);
        const uint32_t qa = ((sbase + L::kQ + u * L::kQTile) & 0x3FFFFu) >> 4;
        const uint32_t ka = ((sbase + L::kK + s * L::kKTile) & 0x3FFFFu) >> 4;
        const uint32_t d = tmem_u + (uint32_t)(u * 128);
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t oq = (uint32_t)((kk / 4) * L::kQHalf + (kk % 4) * 32) >> 4;
          const uint32_t ok = (uint32_t)((kk / 4) * L::kKHalf + (kk % 4) * 32) >> 4;
          umma2_ss_e(d, make_desc(qa + oq + kLbo, kDescHi), make_desc(ka + ok + kLbo, kDescHi), idesc, kk > 0 ? 1u : 0u, ldm);
        }
      };
      auto issue_pv = [&](int u, int s, int kk0, int kk1, bool first) {
        const uint32_t va = ((sbase + L::kV + s * L::kVTile) & 0x3FFFFu) >> 4;
        const uint32_t d = tmem_u + (uint32_t)(256 + u * D);
        const uint32_t a = tmem_u + (uint32_t)(u * 128);
        // A: P_u columns [8kk, 8kk+8) (16 bf16 keys); B: V rows 16kk..16kk+15 of this CTA's 64 columns, MN-major
        for (int kk = kk0; kk < kk1; ++kk)
          umma2_ts_e(d, a + (uint32_t)(kk * 8), make_desc(va + (uint32_t)(kk * 16 * 128 >> 4) + kLbo, kDescHi), idesc_pv,
                     (!first || kk > 0) ? 1u : 0u, ldm);
      };
      uint32_t step = 0;  // K/V tiles consumed so far: tile `step` lives in stage step % kStages
      int k = 0;
      int it = pair;
      int n_pieces = 0;
      if (it < prm.n_items) {
        mbar_wait(BAR(L::LISTFULL + 0), 0);
        n_pieces = uni(s_np[0]);
        // first Q K^T of the first unit
        mbar_wait_cluster(BAR(L::KFULL + 0), 0);
        for (int u = 0; u < 2; ++u) {
          mbar_wait_cluster(BAR(L::QFULL + u), 0);
          ++q_cnt[u];
          tc_fence_after();
          issue_qk(u, 0, min(kPPT, n_pieces));
          umma2_commit_both_e(BAR(L::SFULL + u), ld);
          if (n_pieces <= kPPT) umma2_commit_both_e(BAR(L::QEMPTY + u), ld);
        }
        umma2_commit_both_e(BAR(L::KEMPTY + 0), ld);
      }
      for (; it < prm.n_items; it += n_pairs, ++k) {
        const int buf = k & 1;
        const int n_tiles = (n_pieces + kPPT - 1) / kPPT;
        const bool has_next = it + n_pairs < prm.n_items;
        int n_pieces_next = 0;
        for (int i = 0; i < n_tiles; ++i, ++step) {
          const int vs = (int)(step % L::kStages);
          const int ks = (int)((step + 1) % L::kStages);
          const bool last = (i + 1 == n_tiles);
          const bool more = !last || has_next;  // another Q K^T follows this tile's P V
          int np_next = 0, n_tiles_after = 0;
          if (!last) {
            np_next = min(kPPT, n_pieces - (i + 1) * kPPT);
            n_tiles_after = n_tiles - (i + 2);
          } else if (has_next) {
            mbar_wait(BAR(L::LISTFULL + (buf ^ 1)), (uint32_t)((k + 1) >> 1) & 1u);
            n_pieces_next = uni(s_np[buf ^ 1]);
            np_next = min(kPPT, n_pieces_next);
            n_tiles_after = (n_pieces_next + kPPT - 1) / kPPT - 1;
          }
          const int np = min(kPPT, n_pieces - i * kPPT);
          mbar_wait_cluster(BAR(L::VFULL + vs), (step / L::kStages) & 1u);
          if (more) mbar_wait_cluster(BAR(L::KFULL + ks), ((step + 1) / L::kStages) & 1u);
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            mbar_wait_cluster(BAR(L::PFULL + u), p_cnt[u] & 1u);  // keys 0..63 of P_u, both CTAs
            if (i == 0) {
              // the epilogues of both CTAs have drained the previous unit's O_u
              mbar_wait_cluster(BAR(L::OEMPTY + u), (oe_cnt[u] & 1u) ^ 1u);
              ++oe_cnt[u];
            }
            tc_fence_after();
            issue_pv(u, vs, 0, min(np, kPPT / 2), i == 0);
            mbar_wait_cluster(BAR(L::PFULLB + u), p_cnt[u] & 1u);  // keys 64..127
            ++p_cnt[u];
            tc_fence_after();
            issue_pv(u, vs, kPPT / 2, np, false);
            if (last) umma2_commit_both_e(BAR(L::OFULL + u), ld);
            if (more) {
              if (last) {
                mbar_wait_cluster(BAR(L::QFULL + u), q_cnt[u] & 1u);
                ++q_cnt[u];
                tc_fence_after();
              }
              issue_qk(u, ks, np_next);
              umma2_commit_both_e(BAR(L::SFULL + u), ld);
              if (n_tiles_after == 0) umma2_commit_both_e(BAR(L::QEMPTY + u), ld);  // that was the unit's last Q K^T
            }
          }
          umma2_commit_both_e(BAR(L::VEMPTY + vs), ld);
          if (more) umma2_commit_both_e(BAR(L::KEMPTY + ks), ld);
        }
        if (lane == 0) mbar_arrive(BAR(L::LISTEMPTY + buf));
        n_pieces = n_pieces_next;
      }
      __syncwarp();
    }
  }
  // no CTA of the pair may leave while the other can still signal its barriers or read its shared memory / TMEM
  tc_fence_before();
  cluster_sync_all();
  if (warp == kMmaWarp) {
    tc_fence_after();
    tmem_dealloc2(tmem, 512);
  }
}

}  // namespace

// The CTA-pair kernel covers bf16, head_dim 128, GQA groups of exactly 8 query heads (four 128-row query tiles per
// unit); everything else returns HGA_ERR_UNSUPPORTED and the caller falls back to attend_tc2_kernel.
hga_status launch_attend_pair(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                              void* out, float* lse, cudaStream_t s) {
  using L = SmemP;
  if (!d.bf16_io || d.D != kD || d.G != 8) return HGA_ERR_UNSUPPORTED;
  PairParams prm;
  prm.B = d.B; prm.Hq = d.Hq; prm.Hkv = d.Hkv; prm.N = d.N; prm.n_b = d.n_b; prm.G = d.G;
  prm.jb = d.jb; prm.nj = d.nj;
  prm.F = d.F; prm.L_eff = d.L_eff; prm.gs = d.gs; prm.Kg = d.Kg;
  prm.list_cap = max_key_pieces(d.F, d.L_eff, d.gs, d.Kg);
  prm.scale_log2 = d.scale * 1.4426950408889634f;
  prm.out_bf16 = d.bf16_out ? 1 : 0;
  const long long n_items = (long long)d.B * d.Hkv * d.nj;
  const size_t smem = (size_t)L::kList + 2 * sizeof(int) * (size_t)prm.list_cap;
  if (smem > 227 * 1024 || n_items >= (1ll << 31)) return HGA_ERR_UNSUPPORTED;
  if ((uint64_t)d.B * d.Hq * d.N >= (1ull << 31)) return HGA_ERR_UNSUPPORTED;
  prm.n_items = (int)n_items;
  CUtensorMap tmQ, tmK, tmV, tmO;
  const uint64_t q_rows = (uint64_t)d.B * d.Hq * d.N, kv_rows = (uint64_t)d.B * d.Hkv * d.N;
  bool ok = make_map_2d(&tmQ, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, q, q_rows, kD, 64, 64) &&
            make_map_2d(&tmK, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, k, kv_rows, kD, 64, 16) &&
            make_map_2d(&tmV, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, v, kv_rows, kD, 64, 16);
  ok = ok && (d.bf16_out ? make_map_2d(&tmO, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, out, q_rows, kD, 64, 32)
                         : make_map_2d(&tmO, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, out, q_rows, kD, 32, 32));
  if (!ok) return HGA_ERR_CUDA;
  const int n_sm = current_sm_count();
  if (n_sm <= 0) return HGA_ERR_CUDA;
  HGA_CUDA_OK(cudaFuncSetAttribute(attend_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int n_pairs = (int)(n_items < n_sm / 2 ? n_items : n_sm / 2);
  attend_pair_kernel<<<2 * n_pairs, kThreads, smem, s>>>(tmQ, tmK, tmV, tmO, group_idx, lse, prm);
  return launch_status();
}

}  // namespace hga
