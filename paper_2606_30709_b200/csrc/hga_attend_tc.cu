// S4, tensor-core kernel for bf16 inputs (Eq. (1) PAPER.md:56 over the union set).
//
// One CTA = one (batch, kv head, query block j) unit x up to two 128-row query tiles (a tile = 2 query heads of
// the GQA group x 64 tokens).  The unit's key list (sink, routed groups, local, current chunk) is built in shared
// memory as 16-token pieces; a producer warp gathers K and V pieces with TMA (2-D boxes of 16 rows x 64 bf16,
// 128B swizzle) into a ring of 128-key tiles; one thread issues tcgen05.mma:
//     S_t  = Q_t K^T        (SS: both operands K-major in shared memory, fp32 accumulator in TMEM)
//     O_t += P_t V          (TS: P_t bf16 in TMEM aliasing S_t, V MN-major in shared memory)
// and two softmax warpgroups (one thread per query row) run the online softmax in fp32 straight out of TMEM,
// ping-ponging so that tile 0's softmax overlaps tile 1's MMAs.  The running max is only refreshed (and O rescaled
// in TMEM) when it grows by more than 2^8, which leaves the result mathematically unchanged.
//
// TMEM map (512 columns): S_t at t*128 (P_t overlays its first 64 columns), O_t at 256 + t*D.
#include <cuda.h>
#include <math_constants.h>

#include "hga_common.cuh"
#include "hga_tc_ptx.cuh"

namespace hga {

namespace {

constexpr int kSoftmaxThreads = 256;  // 2 warpgroups
constexpr int kMmaWarp = 8;
constexpr int kLoadWarp = 9;
constexpr int kTcThreads = 320;
constexpr int kTileKeys = 128;        // keys per KV tile (8 pieces)
constexpr int kPiecesPerTile = 8;
constexpr float kRescaleThreshold = 8.0f;  // in log2 units

using namespace tc;


struct TcParams {
  int Hq, Hkv, N, n_b, G;
  int jb;            // first query block of this launch (hga_prefill_window)
  int F, L_eff, gs, Kg;
  int n_mt;          // 128-row query tiles per unit = ceil(G/2)
  int ctas_per_unit; // ceil(n_mt/2)
  int list_cap;
  float scale_log2;  // softmax_scale * log2(e)
  int out_bf16;
};

template <int D>
struct Smem {
  static constexpr int kHalves = D / 64;                  // 64-element (128-byte) column blocks
  static constexpr int kHalfBytes = kTileKeys * 128;      // 128 rows x 128 B = 16 KB
  static constexpr int kTileBytes = kHalves * kHalfBytes; // Q tile / K tile / V tile
  static constexpr int kStages = (D == 128) ? 2 : 4;
  static constexpr int kQ = 0;
  static constexpr int kK = kQ + 2 * kTileBytes;
  static constexpr int kV = kK + kStages * kTileBytes;
  static constexpr int kBar = kV + kStages * kTileBytes;  // mbarriers (8 B each)
  static constexpr int kNumBars = 1 + 4 * kStages + 4;
  static constexpr int kMisc = kBar + 8 * kNumBars;       // tmem base (4 B) + list count (4 B)
  static constexpr int kList = kMisc + 16;
};

template <int D>
__global__ void __launch_bounds__(kTcThreads, 1)
attend_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                 const __grid_constant__ CUtensorMap tmV, const int32_t* __restrict__ group_idx, void* __restrict__ out,
                 float* __restrict__ lse, const TcParams prm) {
  using L = Smem<D>;
  extern __shared__ __align__(1024) unsigned char smem[];
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bar0 = sbase + L::kBar;
  // barrier ids
  auto BAR = [&](int i) { return bar0 + 8u * (uint32_t)i; };
  const int B_QFULL = 0;
  auto B_KFULL = [&](int s) { return 1 + s; };
  auto B_KEMPTY = [&](int s) { return 1 + L::kStages + s; };
  auto B_VFULL = [&](int s) { return 1 + 2 * L::kStages + s; };
  auto B_VEMPTY = [&](int s) { return 1 + 3 * L::kStages + s; };
  auto B_SFULL = [&](int t) { return 1 + 4 * L::kStages + t; };
  auto B_PFULL = [&](int t) { return 1 + 4 * L::kStages + 2 + t; };
  volatile uint32_t* tmem_base_p = reinterpret_cast<volatile uint32_t*>(smem + L::kMisc);
  int* s_count = reinterpret_cast<int*>(smem + L::kMisc + 4);
  int* list = reinterpret_cast<int*>(smem + L::kList);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int j = prm.jb + blockIdx.x / prm.ctas_per_unit;
  const int cu = blockIdx.x % prm.ctas_per_unit;
  const int kv = blockIdx.y, b = blockIdx.z;
  const int mt0 = cu * 2;                               // first query tile of this CTA
  const int nt_cta = min(2, prm.n_mt - mt0);            // query tiles handled here (1 or 2)

  const int32_t* gi = group_idx ? group_idx + (((size_t)b * prm.Hkv + kv) * prm.n_b + j) * prm.Kg : nullptr;
  const int n_pieces = build_key_list(list, s_count, j, prm.F, prm.L_eff, prm.gs, prm.Kg, gi);  // ends with __syncthreads
  const int n_tiles = (n_pieces + kPiecesPerTile - 1) / kPiecesPerTile;
  const int first_cur_piece = n_pieces - kChunk / 16;   // the current chunk's pieces come last

  if (threadIdx.x == 0) {
    mbar_init(BAR(B_QFULL), 1);
    for (int s = 0; s < L::kStages; ++s) {
      mbar_init(BAR(B_KFULL(s)), 1);
      mbar_init(BAR(B_KEMPTY(s)), 1);
      mbar_init(BAR(B_VFULL(s)), 1);
      mbar_init(BAR(B_VEMPTY(s)), 1);
    }
    for (int t = 0; t < 2; ++t) {
      mbar_init(BAR(B_SFULL(t)), 1);
      mbar_init(BAR(B_PFULL(t)), 128);
    }
    fence_barrier_init();
    fence_proxy_async();
  }
  if (warp == kMmaWarp) tmem_alloc(sbase + L::kMisc, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_base_p;

  if (warp == kLoadWarp) {
    // ===================================== TMA producer =====================================================
    const int kv_row0 = (b * prm.Hkv + kv) * prm.N;  // row of token 0 in the flattened [B*Hkv*N, D] K/V matrices
    if (lane == 0) mbar_expect_tx(BAR(B_QFULL), (uint32_t)(nt_cta * L::kTileBytes));
    __syncwarp();
    {
      // Q boxes: (tile t, head-in-tile hh, column block cb) -> 64 rows x 64 columns
      const int nbox = nt_cta * 2 * L::kHalves;
      if (lane < nbox) {
        const int cb = lane % L::kHalves, hh = (lane / L::kHalves) % 2, t = lane / (2 * L::kHalves);
        int head_in_group = (mt0 + t) * 2 + hh;
        if (head_in_group >= prm.G) head_in_group = (mt0 + t) * 2;  // odd G: duplicate a live head, never stored
        const int head = kv * prm.G + head_in_group;
        const int row = (b * prm.Hq + head) * prm.N + j * kChunk;
        tma_load_2d(sbase + L::kQ + t * L::kTileBytes + cb * L::kHalfBytes + hh * 64 * 128, &tmQ, cb * 64, row,
                    BAR(B_QFULL));
      }
    }
    for (int i = 0; i < n_tiles; ++i) {
      const int s = i % L::kStages;
      const uint32_t ph = (uint32_t)(i / L::kStages) & 1u;
      const int np = min(kPiecesPerTile, n_pieces - i * kPiecesPerTile);
      const uint32_t bytes = (uint32_t)(np * 16 * D * 2);
      const int pc = lane / L::kHalves, cb = lane % L::kHalves;
      const bool active = lane < kPiecesPerTile * L::kHalves && pc < np;
      const int row = active ? kv_row0 + list[i * kPiecesPerTile + pc] * 16 : 0;
      const uint32_t off = (uint32_t)(s * L::kTileBytes + cb * L::kHalfBytes + pc * 16 * 128);
      // K tile
      mbar_wait(BAR(B_KEMPTY(s)), ph ^ 1u);
      if (lane == 0) mbar_expect_tx(BAR(B_KFULL(s)), bytes);
      __syncwarp();
      if (active) tma_load_2d(sbase + L::kK + off, &tmK, cb * 64, row, BAR(B_KFULL(s)));
      // V tile
      mbar_wait(BAR(B_VEMPTY(s)), ph ^ 1u);
      if (lane == 0) mbar_expect_tx(BAR(B_VFULL(s)), bytes);
      __syncwarp();
      if (active) tma_load_2d(sbase + L::kV + off, &tmV, cb * 64, row, BAR(B_VFULL(s)));
    }
  } else if (warp == kMmaWarp) {
    // ===================================== MMA issuer (one thread) ==========================================
    if (lane == 0) {
      const uint32_t idesc_pv = umma_idesc(128, D, /*b_mn_major=*/true);
      auto issue_qk = [&](int t, int s, int nkeys) {
        const uint32_t idesc = umma_idesc(128, nkeys, false);
        const uint32_t qa = sbase + L::kQ + t * L::kTileBytes;
        const uint32_t ka = sbase + L::kK + s * L::kTileBytes;
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t o = (uint32_t)((kk / 4) * L::kHalfBytes + (kk % 4) * 32);
          umma_ss(tmem + (uint32_t)(t * 128), umma_desc(qa + o, 16, 1024), umma_desc(ka + o, 16, 1024), idesc,
                  kk > 0 ? 1u : 0u);
        }
      };
      auto issue_pv = [&](int t, int s, int nkeys, bool first) {
        const uint32_t va = sbase + L::kV + s * L::kTileBytes;
        for (int kk = 0; kk < nkeys / 16; ++kk) {
          // A: P_t columns [8kk, 8kk+8) (16 bf16 keys); B: V rows 16kk..16kk+15, MN-major, LBO = next 64 columns
          umma_ts(tmem + (uint32_t)(256 + t * D), tmem + (uint32_t)(t * 128 + kk * 8),
                  umma_desc(va + (uint32_t)(kk * 16 * 128), L::kHalfBytes, 1024), idesc_pv, (!first || kk > 0) ? 1u : 0u);
        }
      };
      auto nkeys_of = [&](int i) { return min(kPiecesPerTile, n_pieces - i * kPiecesPerTile) * 16; };

      mbar_wait(BAR(B_QFULL), 0);
      mbar_wait(BAR(B_KFULL(0)), 0);
      tc_fence_after();
      for (int t = 0; t < nt_cta; ++t) {
        issue_qk(t, 0, nkeys_of(0));
        umma_commit(BAR(B_SFULL(t)));
      }
      umma_commit(BAR(B_KEMPTY(0)));
      for (int i = 0; i < n_tiles; ++i) {
        const int vs = i % L::kStages;
        const int ks = (i + 1) % L::kStages;
        const bool more = i + 1 < n_tiles;
        mbar_wait(BAR(B_VFULL(vs)), (uint32_t)(i / L::kStages) & 1u);
        if (more) mbar_wait(BAR(B_KFULL(ks)), (uint32_t)((i + 1) / L::kStages) & 1u);
        for (int t = 0; t < nt_cta; ++t) {
          mbar_wait(BAR(B_PFULL(t)), (uint32_t)i & 1u);
          tc_fence_after();
          issue_pv(t, vs, nkeys_of(i), i == 0);
          if (more) issue_qk(t, ks, nkeys_of(i + 1));
          umma_commit(BAR(B_SFULL(t)));  // S_t(i+1) ready and O_t quiescent  /  final: O_t complete
        }
        umma_commit(BAR(B_VEMPTY(vs)));
        if (more) umma_commit(BAR(B_KEMPTY(ks)));
      }
    }
    __syncwarp();
  } else {
    // ===================================== softmax warpgroups ===============================================
    const int t = warp / 4;  // query tile of this warpgroup
    if (t < nt_cta) {
      const int row = (warp % 4) * 32 + lane;          // row of the 128-row tile == TMEM lane
      const uint32_t lane_base = (uint32_t)((warp % 4) * 32) << 16;
      const uint32_t s_addr = tmem + lane_base + (uint32_t)(t * 128);
      const uint32_t o_addr = tmem + lane_base + (uint32_t)(256 + t * D);
      const int q_pos = j * kChunk + (row % 64);
      const float sl2 = prm.scale_log2;
      float m_run = -CUDART_INF_F;  // running reference max, raw logit units
      float l_run = 0.f;
      for (int i = 0; i < n_tiles; ++i) {
        const int np = min(kPiecesPerTile, n_pieces - i * kPiecesPerTile);
        const bool masked = (i * kPiecesPerTile + np > first_cur_piece) || np < kPiecesPerTile;
        mbar_wait(BAR(B_SFULL(t)), (uint32_t)i & 1u);
        tc_fence_after();
        uint32_t sr[128];
        tmem_ld32(s_addr + 0, sr + 0);
        tmem_ld32(s_addr + 32, sr + 32);
        tmem_ld32(s_addr + 64, sr + 64);
        tmem_ld32(s_addr + 96, sr + 96);
        tmem_wait_ld();
        if (masked) {
#pragma unroll
          for (int pc = 0; pc < kPiecesPerTile; ++pc) {
            const int kp0 = (pc < np) ? list[i * kPiecesPerTile + pc] * 16 : 0x3fffffff;
#pragma unroll
            for (int e = 0; e < 16; ++e)
              if (kp0 + e > q_pos) sr[pc * 16 + e] = __float_as_uint(-CUDART_INF_F);  // causal / beyond the tile
          }
        }
        float mx = __uint_as_float(sr[0]);
#pragma unroll
        for (int c = 1; c < 128; ++c) mx = fmaxf(mx, __uint_as_float(sr[c]));
        const float m_new = fmaxf(m_run, mx);
        const bool need = (m_new - m_run) * sl2 > kRescaleThreshold;  // first tile: +inf > 8
        if (__any_sync(0xffffffffu, need)) {
          float alpha = 1.f;
          if (need) {
            alpha = (m_run == -CUDART_INF_F) ? 0.f : fast_exp2((m_run - m_new) * sl2);
            m_run = m_new;
            l_run *= alpha;
          }
          if (i > 0) {
            // O_t is quiescent here: S_FULL(i) was committed after PV(t, i-1)
#pragma unroll
            for (int c0 = 0; c0 < D; c0 += 32) {
              uint32_t orr[32];
              tmem_ld32(o_addr + c0, orr);
              tmem_wait_ld();
#pragma unroll
              for (int c = 0; c < 32; ++c) orr[c] = __float_as_uint(__uint_as_float(orr[c]) * alpha);
              tmem_st32(o_addr + c0, orr);
            }
          }
        }
        const float m_use = (m_run == -CUDART_INF_F) ? 0.f : m_run;
        const float neg_m = -m_use * sl2;
        float lsum = 0.f;
#pragma unroll
        for (int c0 = 0; c0 < 128; c0 += 32) {
          uint32_t pr[16];
#pragma unroll
          for (int c = 0; c < 16; ++c) {
            const float p0 = fast_exp2(fmaf(__uint_as_float(sr[c0 + 2 * c]), sl2, neg_m));
            const float p1 = fast_exp2(fmaf(__uint_as_float(sr[c0 + 2 * c + 1]), sl2, neg_m));
            __nv_bfloat162 h = __floats2bfloat162_rn(p0, p1);  // .x (low half) = key 2c, .y = key 2c+1
            const uint32_t u = *reinterpret_cast<uint32_t*>(&h);
            pr[c] = u;
            // the denominator sums the SAME rounded weights the PV MMA multiplies
            lsum += __uint_as_float(u << 16) + __uint_as_float(u & 0xffff0000u);
          }
          if (c0 < np * 16) tmem_st16(s_addr + (uint32_t)(c0 / 2), pr);  // P overlays S (already in registers)
        }
        l_run += lsum;
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(BAR(B_PFULL(t)));
      }
      // ---- epilogue: O_t / l -> global -----------------------------------------------------------------------
      mbar_wait(BAR(B_SFULL(t)), (uint32_t)n_tiles & 1u);
      tc_fence_after();
      const int head_in_group = (mt0 + t) * 2 + row / 64;
      const bool live = head_in_group < prm.G;
      const int head = kv * prm.G + (live ? head_in_group : 0);
      const size_t orow = ((size_t)b * prm.Hq + head) * prm.N + (size_t)j * kChunk + (row % 64);
      const float inv = 1.f / l_run;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t orr[32];
        tmem_ld32(o_addr + c0, orr);
        tmem_wait_ld();
        if (live) {
          if (prm.out_bf16) {
            __nv_bfloat16* dst = reinterpret_cast<__nv_bfloat16*>(out) + orow * D + c0;
#pragma unroll
            for (int c = 0; c < 32; c += 8) {
              uint32_t w[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                __nv_bfloat162 h = __floats2bfloat162_rn(__uint_as_float(orr[c + 2 * e]) * inv,
                                                         __uint_as_float(orr[c + 2 * e + 1]) * inv);
                w[e] = *reinterpret_cast<uint32_t*>(&h);
              }
              *reinterpret_cast<uint4*>(dst + c) = make_uint4(w[0], w[1], w[2], w[3]);
            }
          } else {
            float* dst = reinterpret_cast<float*>(out) + orow * D + c0;
#pragma unroll
            for (int c = 0; c < 32; c += 4)
              *reinterpret_cast<float4*>(dst + c) =
                  make_float4(__uint_as_float(orr[c]) * inv, __uint_as_float(orr[c + 1]) * inv,
                              __uint_as_float(orr[c + 2]) * inv, __uint_as_float(orr[c + 3]) * inv);
          }
        }
      }
      if (lse != nullptr && live) lse[orow] = (m_run * sl2 + log2f(l_run)) * 0.69314718055994530942f;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kMmaWarp) {
    tc_fence_after();
    tmem_dealloc(tmem, 512);
  }
}

// ---- host side ------------------------------------------------------------------------------------------------
bool make_map(CUtensorMap* m, const void* base, uint64_t rows, int D, int box_rows) {
  return make_map_2d(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, base, rows, D, 64, box_rows);
}

template <int D>
hga_status launch_tc_t(const Derived& d, const void* q, const void* k, const void* v, const int32_t* gi, void* out,
                       float* lse, cudaStream_t s) {
  using L = Smem<D>;
  TcParams prm;
  prm.Hq = d.Hq; prm.Hkv = d.Hkv; prm.N = d.N; prm.n_b = d.n_b; prm.G = d.G;
  prm.jb = d.jb;
  prm.F = d.F; prm.L_eff = d.L_eff; prm.gs = d.gs; prm.Kg = d.Kg;
  prm.n_mt = (d.G + 1) / 2;
  prm.ctas_per_unit = (prm.n_mt + 1) / 2;
  prm.list_cap = max_key_pieces(d.F, d.L_eff, d.gs, d.Kg);
  prm.scale_log2 = d.scale * 1.4426950408889634f;
  prm.out_bf16 = d.bf16_out ? 1 : 0;
  const size_t smem = (size_t)L::kList + sizeof(int) * (size_t)prm.list_cap + 1024;  // + slack for 1024-B alignment
  if (smem > 227 * 1024) return HGA_ERR_UNSUPPORTED;
  if ((uint64_t)d.B * d.Hq * d.N >= (1ull << 31)) return HGA_ERR_UNSUPPORTED;
  CUtensorMap tmQ, tmK, tmV;
  if (!make_map(&tmQ, q, (uint64_t)d.B * d.Hq * d.N, D, 64) || !make_map(&tmK, k, (uint64_t)d.B * d.Hkv * d.N, D, 16) ||
      !make_map(&tmV, v, (uint64_t)d.B * d.Hkv * d.N, D, 16))
    return HGA_ERR_CUDA;
  auto kern = attend_tc_kernel<D>;
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(d.nj * prm.ctas_per_unit, d.Hkv, d.B);
  kern<<<grid, kTcThreads, smem, s>>>(tmQ, tmK, tmV, gi, out, lse, prm);
  return launch_status();
}

}  // namespace

hga_status launch_attend_tc(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                            void* out, float* lse, cudaStream_t s) {
  if (!d.bf16_io) return HGA_ERR_UNSUPPORTED;
  return d.D == 128 ? launch_tc_t<128>(d, q, k, v, group_idx, out, lse, s) : launch_tc_t<64>(d, q, k, v, group_idx, out, lse, s);
}

}  // namespace hga
