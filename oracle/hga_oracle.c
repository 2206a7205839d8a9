/*
 * hga_oracle.c -- CPU ORACLE for Hierarchical Global Attention (HGA) prefill.
 *
 * THIS FILE IS TEST INFRASTRUCTURE.  It is a plain, slow, fp64 restatement of what the paper
 * (arxiv/paper_2606_30709, /root/reference/PAPER.md) says the method computes.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
 * code, header, table or helper with the CUDA path under paper_2606_30709_b200/.
 *
 * The method is "a heuristic selection followed by an exact computation", so the
 * oracle follows the algorithm step by step in the paper's order:
 *   O1 RoPE                         PAPER.md:62   (section 2, "RoPE")
 *   O2 mixed-RoPE summaries         PAPER.md:80-89 (section 3.2)
 *   O3 chunk-shared pooled query
 *   O4 deterministic visibility +
 *      chunk-level content routing  PAPER.md:95-97 (section 3.3)
 *   O5 group-level refinement
 *   O6 exact-token softmax attention over the union set   PAPER.md:103-109 (section 3.4), Eq. (1)
 * Readings of points the paper leaves open (R1..R16) are listed in DESIGN.md; each is marked below.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): full coverage == dense causal attention Eq. (1)
 * (PAPER.md:281); top-k == brute-force sort; softmax rows sum to 1; union set contains sink/local/current
 * and has the paper's printed sizes; summary closed forms; RoPE relative-position
 * invariance.  PARITY UNPINNED: the *choices* R1 (which pairs are high-frequency), R2 (middle position) and
 * R4 (how a 64-query block becomes one routing score) -- the paper prints no worked example for them.
 *
 * All tensors handled here are ONE (batch, kv-head) slice: q [G,N,D], k [N,D], v [N,D].  No blocking,
 * fusion or reordering beyond what the definitions state.  OpenMP only parallelises independent blocks.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define HGA_ORACLE_OK 0
#define HGA_ORACLE_ERR_ARG 1
#define HGA_ORACLE_ERR_NONFINITE 2
#define HGA_ORACLE_ERR_INDEX 3

typedef struct {
  int32_t G;          /* query heads per KV head (GQA group size) */
  int32_t N;          /* sequence length of the slice */
  int32_t D;          /* head dim (even) */
  int32_t C;          /* chunk length */
  int32_t gs;         /* group length g_s */
  int32_t F;          /* sink chunks ("keep first") */
  int32_t L;          /* local chunks ("keep last") */
  int32_t Kc;         /* chunk route budget K_c */
  int32_t Kg;         /* group route budget K_g */
  int32_t n_hi_chunk; /* # leading (highest-frequency) RoPE pairs using "rotate then average" at chunk level */
  int32_t n_hi_group; /* same at group level.  -1 = default rule R1 */
  int32_t io_bf16;    /* 1: Q_rot/K_rot are stored as bf16 (RNE) before attention; 0: as fp32 (R7) */
  int64_t pos0;       /* position of token 0 */
  double base;        /* RoPE base */
  double scale;       /* softmax scale; <= 0 -> 1/sqrt(D) (Eq. 1) */
  int64_t pos_mod;    /* N3 variant: RoPE position index wrapped, p <- p mod pos_mod (the paper uses
                         65536); 0 = off.  Reading R18: every position that enters a rotation is wrapped, and
                         pos_mod and pos0 must be multiples of C so that no span straddles a wrap (its "middle
                         position" R2 is then wrapped start + (S-1)/2); the routing algorithm is unchanged. */
  int32_t route_max;  /* N3 variant (R4's alternative): 0 = a block's score of a candidate is the
                         dot product with the POOLED query (mean of per-query scores); 1 = the MAX over the block's
                         64*G per-query scores.  Reading R19: the per-query scores use the rotated queries as STORED
                         (rounded to the I/O dtype, the only per-query rotated form the method keeps, R7); the pooled
                         query is still returned.  Everything downstream (top-k, ties, order) is unchanged. */
  int32_t pad_;
} hga_oracle_params;

int hga_oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------------ */
/* O1  RoPE.  Reading R6: half-split pairing (x[i], x[i+D/2]), theta_i = base^(-2i/D).  */
/* ------------------------------------------------------------------------------------------------ */
double hga_oracle_theta(int D, double base, int i) { return pow(base, -2.0 * (double)i / (double)D); }

/* rotate one pair (a,b) by angle ang: (a cos - b sin, b cos + a sin) */
static void rot_pair(double a, double b, double ang, double* oa, double* ob) {
  double c = cos(ang), s = sin(ang);
  *oa = a * c - b * s;
  *ob = b * c + a * s;
}

/* N3: the position index that enters a rotation, p <- p mod pos_mod; pos_mod = 0 leaves p as is */
static int64_t wrap_pos(int64_t p, int64_t pos_mod) { return pos_mod > 0 ? p % pos_mod : p; }

/* x [n_rows, D] fp32; row r sits at position pos_first + r (wrapped modulo pos_mod if > 0).  out [n_rows, D] fp64. */
int hga_oracle_rope_mod(const float* x, int n_rows, int D, int64_t pos_first, int64_t pos_mod, double base,
                        double* out) {
  if (D <= 0 || (D & 1) || pos_mod < 0 || pos_first < 0) return HGA_ORACLE_ERR_ARG;
  int half = D / 2;
  for (int r = 0; r < n_rows; ++r) {
    double p = (double)wrap_pos(pos_first + r, pos_mod);
    for (int i = 0; i < half; ++i) {
      double th = hga_oracle_theta(D, base, i);
      rot_pair((double)x[(size_t)r * D + i], (double)x[(size_t)r * D + i + half], p * th,
               &out[(size_t)r * D + i], &out[(size_t)r * D + i + half]);
    }
  }
  return HGA_ORACLE_OK;
}

int hga_oracle_rope(const float* x, int n_rows, int D, int64_t pos_first, double base, double* out) {
  return hga_oracle_rope_mod(x, n_rows, D, pos_first, 0, base, out);
}

/* Storage rounding R7: round fp64 -> nearest fp32, or nearest bf16 (ties to even), in ONE rounding. */
static double round_to_bf16(double x) {
  if (x == 0.0 || !isfinite(x)) return x;
  int e;
  double m = frexp(x, &e);          /* x = m * 2^e, 0.5 <= |m| < 1 */
  double q = nearbyint(ldexp(m, 8)); /* keep 8 significant bits (bf16: 1 implicit + 7 stored); RNE mode */
  return ldexp(q, e - 8);            /* magnitudes here are far from bf16's subnormal/overflow range */
}
void hga_oracle_round_io(double* x, size_t n, int io_bf16) {
  for (size_t i = 0; i < n; ++i) x[i] = io_bf16 ? round_to_bf16(x[i]) : (double)(float)x[i];
}

/* ------------------------------------------------------------------------------------------------ */
/* O2  Mixed-RoPE routing summaries.                                                 */
/*     R1: pair i is "high-frequency" iff i < n_hi; default n_hi = #{i : 2*pi/theta_i <= span}.       */
/*     R2: "middle position" = start + (S-1)/2.   R3: mean (not sum).                                 */
/* ------------------------------------------------------------------------------------------------ */
int hga_oracle_default_n_hi(int D, double base, int span) {
  int n = 0;
  for (int i = 0; i < D / 2; ++i)
    if (2.0 * M_PI / hga_oracle_theta(D, base, i) <= (double)span) ++n;
  return n;
}

/* N3 variants of R1 (the paper gives no threshold): which pairs are "high-frequency" for a span of
   S tokens.  rule 0: wavelength 2*pi/theta_i <= S (the default above); rule 1: the span sweeps at least half a turn,
   theta_i * S >= pi; rule 2: the span sweeps at least one radian, theta_i * S >= 1.  theta_i decreases with i, so
   each rule selects a leading block of pairs and the count is all a caller needs (passed as n_hi). */
int hga_oracle_n_hi_rule(int D, double base, int span, int rule) {
  int n = 0;
  for (int i = 0; i < D / 2; ++i) {
    double th = hga_oracle_theta(D, base, i);
    int hi = rule == 0 ? (2.0 * M_PI / th <= (double)span)
           : rule == 1 ? (th * (double)span >= M_PI)
           : rule == 2 ? (th * (double)span >= 1.0) : 0;
    if (hi) ++n;
  }
  return (rule < 0 || rule > 2) ? -1 : n;
}

/* k_raw [N,D] fp32 (un-rotated keys); spans of S tokens; out [N/S, D] fp64. */
int hga_oracle_summaries_mod(const float* k_raw, int N, int D, int S, int n_hi, int64_t pos0, int64_t pos_mod,
                             double base, double* out) {
  if (S <= 0 || N % S || (D & 1) || pos_mod < 0 || pos0 < 0) return HGA_ORACLE_ERR_ARG;
  if (pos_mod > 0 && (pos_mod % S || pos0 % S)) return HGA_ORACLE_ERR_ARG; /* R18: no span straddles a wrap */
  int half = D / 2;
  if (n_hi < 0) n_hi = hga_oracle_default_n_hi(D, base, S);
  if (n_hi > half) return HGA_ORACLE_ERR_ARG;
  for (int sp = 0; sp < N / S; ++sp) {
    int start = sp * S;
    double p_mid = (double)wrap_pos(pos0 + start, pos_mod) + 0.5 * (double)(S - 1);
    for (int i = 0; i < half; ++i) {
      double th = hga_oracle_theta(D, base, i);
      double sa = 0.0, sb = 0.0;
      if (i < n_hi) {
        /* high-frequency pair: rotate per token, then average */
        for (int t = 0; t < S; ++t) {
          double ra, rb;
          const float* row = k_raw + (size_t)(start + t) * D;
          rot_pair((double)row[i], (double)row[i + half], (double)wrap_pos(pos0 + start + t, pos_mod) * th,
                   &ra, &rb);
          sa += ra;
          sb += rb;
        }
        sa /= (double)S;
        sb /= (double)S;
      } else {
        /* low-frequency pair: average raw keys, then rotate at the middle position */
        double ma = 0.0, mb = 0.0;
        for (int t = 0; t < S; ++t) {
          const float* row = k_raw + (size_t)(start + t) * D;
          ma += (double)row[i];
          mb += (double)row[i + half];
        }
        ma /= (double)S;
        mb /= (double)S;
        rot_pair(ma, mb, p_mid * th, &sa, &sb);
      }
      out[(size_t)sp * D + i] = sa;
      out[(size_t)sp * D + i + half] = sb;
    }
  }
  return HGA_ORACLE_OK;
}

int hga_oracle_summaries(const float* k_raw, int N, int D, int S, int n_hi, int64_t pos0, double base,
                         double* out) {
  return hga_oracle_summaries_mod(k_raw, N, D, S, n_hi, pos0, 0, base, out);
}

/* ------------------------------------------------------------------------------------------------ */
/* O3  Chunk-shared pooled query (R4/R5): mean of the rotated (un-rounded) queries over the block's C   */
/*     tokens and the G heads of the KV group.  q_rot [G,N,D] fp64 -> qbar [N/C, D].                   */
/* ------------------------------------------------------------------------------------------------ */
int hga_oracle_pool_queries(const double* q_rot, int G, int N, int D, int C, double* qbar) {
  if (C <= 0 || N % C) return HGA_ORACLE_ERR_ARG;
  for (int j = 0; j < N / C; ++j)
    for (int d = 0; d < D; ++d) {
      double s = 0.0;
      for (int h = 0; h < G; ++h)
        for (int t = 0; t < C; ++t) s += q_rot[((size_t)h * N + (size_t)j * C + t) * D + d];
      qbar[(size_t)j * D + d] = s / (double)(G * C);
    }
  return HGA_ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------ */
/* Top-k by (score descending, index ascending) -- R8.  Plain selection: k passes over the candidates. */
/* cand_idx/cand_score: n candidates.  Writes min(k,n) winners in ASCENDING INDEX order; returns count. */
/* ------------------------------------------------------------------------------------------------ */
static int topk_select(const int* cand_idx, const double* cand_score, int n, int k, int* out_idx,
                       double* out_score) {
  int take = k < n ? k : n;
  char* used = (char*)calloc((size_t)(n > 0 ? n : 1), 1);
  int* win = (int*)malloc(sizeof(int) * (size_t)(take > 0 ? take : 1));
  for (int s = 0; s < take; ++s) {
    int best = -1;
    for (int c = 0; c < n; ++c) {
      if (used[c]) continue;
      if (best < 0 || cand_score[c] > cand_score[best] ||
          (cand_score[c] == cand_score[best] && cand_idx[c] < cand_idx[best]))
        best = c;
    }
    used[best] = 1;
    win[s] = best;
  }
  /* ascending index order (insertion sort on the winners) */
  for (int a = 1; a < take; ++a) {
    int w = win[a], b = a - 1;
    while (b >= 0 && cand_idx[win[b]] > cand_idx[w]) {
      win[b + 1] = win[b];
      --b;
    }
    win[b + 1] = w;
  }
  for (int s = 0; s < take; ++s) {
    out_idx[s] = cand_idx[win[s]];
    if (out_score) out_score[s] = cand_score[win[s]];
  }
  free(used);
  free(win);
  return take;
}

static double dot(const double* a, const double* b, int D) {
  double s = 0.0;
  for (int d = 0; d < D; ++d) s += a[d] * b[d];
  return s;
}

/* ------------------------------------------------------------------------------------------------ */
/* O4  Chunk routing for block j.                                                   */
/*     L_eff = max(L,1): the immediately preceding chunk is force-included (R14).                     */
/*     Middle candidates M_j = {F, ..., j - L_eff - 1}; score(c) = qbar . S_c[c] (raw dot, R11);       */
/*     keep the min(K_c, |M_j|) best (R9); ties -> lower index; ascending output, -1 padded (R8).      */
/*     all_scores (optional, [n_b]) receives score(c) for c in M_j and NaN elsewhere.                  */
/* ------------------------------------------------------------------------------------------------ */
int hga_oracle_route_chunks(const double* qbar_j, const double* S_c, int n_b, int D, int j, int F, int L,
                            int Kc, int* idx_out, double* score_out, double* all_scores) {
  int L_eff = L > 1 ? L : 1;
  int lo = F, hi = j - L_eff; /* candidates c in [lo, hi) */
  int n = hi > lo ? hi - lo : 0;
  int* ci = (int*)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
  double* cs = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  if (all_scores)
    for (int c = 0; c < n_b; ++c) all_scores[c] = NAN;
  for (int c = 0; c < n; ++c) {
    ci[c] = lo + c;
    cs[c] = dot(qbar_j, S_c + (size_t)(lo + c) * D, D);
    if (all_scores) all_scores[lo + c] = cs[c];
  }
  for (int s = 0; s < Kc; ++s) {
    idx_out[s] = -1;
    if (score_out) score_out[s] = 0.0;
  }
  int cnt = topk_select(ci, cs, n, Kc, idx_out, score_out);
  free(ci);
  free(cs);
  return cnt;
}

/* ------------------------------------------------------------------------------------------------ */
/* O5  Group refinement: candidates = the C/g_s groups of every selected chunk;          */
/*     score(g) = qbar . S_g[g] (group score alone, R10); one global top-K_g; ascending, -1 padded.     */
/*     cand_scores (optional, [n_chunks * C/gs]) receives the candidates' scores in candidate order.   */
/* ------------------------------------------------------------------------------------------------ */
int hga_oracle_route_groups(const double* qbar_j, const double* S_g, int D, int gpc, const int* chunk_idx,
                            int n_chunks, int Kg, int* idx_out, double* score_out, double* cand_scores) {
  int n = n_chunks * gpc;
  int* ci = (int*)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
  double* cs = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  for (int a = 0; a < n_chunks; ++a)
    for (int u = 0; u < gpc; ++u) {
      int g = chunk_idx[a] * gpc + u;
      ci[a * gpc + u] = g;
      cs[a * gpc + u] = dot(qbar_j, S_g + (size_t)g * D, D);
      if (cand_scores) cand_scores[a * gpc + u] = cs[a * gpc + u];
    }
  for (int s = 0; s < Kg; ++s) {
    idx_out[s] = -1;
    if (score_out) score_out[s] = 0.0;
  }
  int cnt = topk_select(ci, cs, n, Kg, idx_out, score_out);
  free(ci);
  free(cs);
  return cnt;
}

/* ------------------------------------------------------------------------------------------------ */
/* N3  R4's alternative: max over per-query scores (PAPER.md:33, 45, 97 leave open how the 64*G queries of a   */
/*     block become one score).  q_rows [n_rows, D] are the block's rotated queries (all heads of the GQA      */
/*     group); score(c) = max_r q_rows[r] . S[c].  Candidate sets, budgets, ties and output order are those of */
/*     O4 / O5.                                                                                              */
/* ------------------------------------------------------------------------------------------------ */
static double max_dot(const double* q_rows, int n_rows, const double* s, int D) {
  double best = -INFINITY;
  for (int r = 0; r < n_rows; ++r) {
    double v = dot(q_rows + (size_t)r * D, s, D);
    if (v > best) best = v;
  }
  return best;
}

int hga_oracle_route_chunks_max(const double* q_rows, int n_rows, const double* S_c, int n_b, int D, int j, int F,
                                int L, int Kc, int* idx_out, double* score_out, double* all_scores) {
  int L_eff = L > 1 ? L : 1;
  int lo = F, hi = j - L_eff; /* candidates c in [lo, hi) */
  int n = hi > lo ? hi - lo : 0;
  int* ci = (int*)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
  double* cs = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  if (n_rows <= 0) { free(ci); free(cs); return -1; }
  if (all_scores)
    for (int c = 0; c < n_b; ++c) all_scores[c] = NAN;
  for (int c = 0; c < n; ++c) {
    ci[c] = lo + c;
    cs[c] = max_dot(q_rows, n_rows, S_c + (size_t)(lo + c) * D, D);
    if (all_scores) all_scores[lo + c] = cs[c];
  }
  for (int s = 0; s < Kc; ++s) {
    idx_out[s] = -1;
    if (score_out) score_out[s] = 0.0;
  }
  int cnt = topk_select(ci, cs, n, Kc, idx_out, score_out);
  free(ci);
  free(cs);
  return cnt;
}

int hga_oracle_route_groups_max(const double* q_rows, int n_rows, const double* S_g, int D, int gpc,
                                const int* chunk_idx, int n_chunks, int Kg, int* idx_out, double* score_out,
                                double* cand_scores) {
  int n = n_chunks * gpc;
  int* ci = (int*)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
  double* cs = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  if (n_rows <= 0) { free(ci); free(cs); return -1; }
  for (int a = 0; a < n_chunks; ++a)
    for (int u = 0; u < gpc; ++u) {
      int g = chunk_idx[a] * gpc + u;
      ci[a * gpc + u] = g;
      cs[a * gpc + u] = max_dot(q_rows, n_rows, S_g + (size_t)g * D, D);
      if (cand_scores) cand_scores[a * gpc + u] = cs[a * gpc + u];
    }
  for (int s = 0; s < Kg; ++s) {
    idx_out[s] = -1;
    if (score_out) score_out[s] = 0.0;
  }
  int cnt = topk_select(ci, cs, n, Kg, idx_out, score_out);
  free(ci);
  free(cs);
  return cnt;
}

/* ------------------------------------------------------------------------------------------------ */
/* Union token set of block j (R13: set union):                                      */
/*   sink chunks {0..min(F,j)-1}  U  local chunks {max(0,j-L_eff)..j-1}  U  tokens of the opened groups */
/*   U  current chunk (the causal cut u <= t is applied per query row in O6).                          */
/* visible [ (j+1)*C ] bytes: 1 = token belongs to the set.  Returns an error for a group that is not a  */
/* closed earlier group (index < 0 other than the -1 pad, or reaching into chunk j or later) or that    */
/* appears twice in the list.                                                                          */
/* ------------------------------------------------------------------------------------------------ */
int hga_oracle_key_set(int j, int C, int gs, int F, int L, const int* group_idx, int n_group_slots,
                       unsigned char* visible) {
  int L_eff = L > 1 ? L : 1;
  int n_tok = (j + 1) * C;
  memset(visible, 0, (size_t)n_tok);
  for (int c = 0; c < F && c < j; ++c)
    for (int t = 0; t < C; ++t) visible[c * C + t] = 1;
  for (int c = (j - L_eff > 0 ? j - L_eff : 0); c < j; ++c)
    for (int t = 0; t < C; ++t) visible[c * C + t] = 1;
  unsigned char* seen = (unsigned char*)calloc((size_t)(n_tok / gs + 1), 1);
  for (int s = 0; s < n_group_slots; ++s) {
    int g = group_idx[s];
    if (g == -1) continue;
    if (g < 0 || (g + 1) * gs > j * C || seen[g]) {
      free(seen);
      return HGA_ORACLE_ERR_INDEX;
    }
    seen[g] = 1;
    for (int t = 0; t < gs; ++t) visible[g * gs + t] = 1;
  }
  free(seen);
  for (int t = 0; t < C; ++t) visible[j * C + t] = 1;
  return HGA_ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------ */
/* O6  Exact-token attention for block j (Eq. (1) PAPER.md:56 restricted to the set). */
/*   q_blk [G,C,D]: rotated queries of block j, already rounded to the storage type (R7)               */
/*   k_rot [N,D], v [N,D]: rotated+rounded keys, values as given (fp64 copies)                         */
/*   out [G,C,D], lse [G,C] (natural log of the softmax denominator, incl. the max), n_keys [C] optional */
/* ------------------------------------------------------------------------------------------------ */
/* Rows [r0, r0+W) of block j: q_rows [G,W,D]; k_rot / v hold at least the tokens 0 .. j*C+r0+W-1.      */
/* out [G,W,D], lse [G,W], n_keys [W] optional.  hga_oracle_attend_block is the case r0 = 0, W = C.     */
int hga_oracle_attend_rows(const double* q_rows, const double* k_rot, const double* v, int G, int n_tok_avail,
                           int D, int C, int gs, int F, int L, int j, int r0, int W, const int* group_idx,
                           int n_group_slots, double scale, double* out, double* lse, int* n_keys) {
  if (r0 < 0 || W < 0 || r0 + W > C || j * C + r0 + W > n_tok_avail) return HGA_ORACLE_ERR_ARG;
  if (scale <= 0.0) scale = 1.0 / sqrt((double)D);
  int n_tok = (j + 1) * C;
  unsigned char* vis = (unsigned char*)malloc((size_t)n_tok);
  int rc = hga_oracle_key_set(j, C, gs, F, L, group_idx, n_group_slots, vis);
  if (rc) {
    free(vis);
    return rc;
  }
  double* logit = (double*)malloc(sizeof(double) * (size_t)n_tok);
  for (int h = 0; h < G; ++h)
    for (int r = 0; r < W; ++r) {
      const double* q = q_rows + ((size_t)h * W + r) * D;
      int t = j * C + r0 + r; /* query token; keys u <= t only (causal, Eq. 1) */
      double m = -INFINITY;
      int cnt = 0;
      for (int u = 0; u <= t; ++u) {
        if (!vis[u]) continue;
        logit[u] = scale * dot(q, k_rot + (size_t)u * D, D);
        if (logit[u] > m) m = logit[u];
        ++cnt;
      }
      double den = 0.0;
      double* o = out + ((size_t)h * W + r) * D;
      for (int d = 0; d < D; ++d) o[d] = 0.0;
      for (int u = 0; u <= t; ++u) {
        if (!vis[u]) continue;
        double w = exp(logit[u] - m); /* max-subtracted softmax numerator */
        den += w;
        for (int d = 0; d < D; ++d) o[d] += w * v[(size_t)u * D + d];
      }
      for (int d = 0; d < D; ++d) o[d] /= den;
      if (lse) lse[(size_t)h * W + r] = m + log(den);
      if (n_keys && h == 0) n_keys[r] = cnt;
    }
  free(logit);
  free(vis);
  return HGA_ORACLE_OK;
}

int hga_oracle_attend_block(const double* q_blk, const double* k_rot, const double* v, int G, int N, int D,
                            int C, int gs, int F, int L, int j, const int* group_idx, int n_group_slots,
                            double scale, double* out, double* lse, int* n_keys) {
  if ((j + 1) * C > N) return HGA_ORACLE_ERR_ARG;
  return hga_oracle_attend_rows(q_blk, k_rot, v, G, N, D, C, gs, F, L, j, 0, C, group_idx, n_group_slots, scale,
                                out, lse, n_keys);
}

/* Dense causal attention, Eq. (1), for the rows of block j: every token u <= t is a key.  */
/* This is the paper's baseline; tests compare it with an independent numpy Eq. (1).     */
int hga_oracle_dense_block(const double* q_blk, const double* k_rot, const double* v, int G, int N, int D,
                           int C, int j, double scale, double* out, double* lse) {
  if ((j + 1) * C > N) return HGA_ORACLE_ERR_ARG;
  if (scale <= 0.0) scale = 1.0 / sqrt((double)D);
  double* logit = (double*)malloc(sizeof(double) * (size_t)((j + 1) * C));
  for (int h = 0; h < G; ++h)
    for (int r = 0; r < C; ++r) {
      const double* q = q_blk + ((size_t)h * C + r) * D;
      int t = j * C + r;
      double m = -INFINITY;
      for (int u = 0; u <= t; ++u) {
        logit[u] = scale * dot(q, k_rot + (size_t)u * D, D);
        if (logit[u] > m) m = logit[u];
      }
      double den = 0.0;
      double* o = out + ((size_t)h * C + r) * D;
      for (int d = 0; d < D; ++d) o[d] = 0.0;
      for (int u = 0; u <= t; ++u) {
        double w = exp(logit[u] - m);
        den += w;
        for (int d = 0; d < D; ++d) o[d] += w * v[(size_t)u * D + d];
      }
      for (int d = 0; d < D; ++d) o[d] /= den;
      if (lse) lse[(size_t)h * C + r] = m + log(den);
    }
  free(logit);
  return HGA_ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------ */
/* Whole pipeline for one (batch, kv-head) slice, steps O1..O6 in order, for a list of query blocks.   */
/* Every output pointer may be NULL.  Buffers:                                                         */
/*   q_raw [G,N,D] f32, k_raw [N,D] f32, v [N,D] f32 (values already in the storage type)               */
/*   blocks [n_blocks] block ids j (NULL -> 0..n_blocks-1)                                             */
/*   k_rot_io [N,D]: rotated keys after storage rounding;  chunk_sum [N/C,D];  group_sum [N/gs,D]       */
/*   q_pooled [n_blocks,D];  chunk_idx/score [n_blocks,Kc];  n_chunks [n_blocks];                       */
/*   chunk_all_scores [n_blocks, N/C] (NaN = not a candidate);                                          */
/*   group_idx/score [n_blocks,Kg];  n_groups [n_blocks];  group_cand_scores [n_blocks, Kc*C/gs]        */
/*   out [n_blocks,G,C,D];  lse [n_blocks,G,C]                                                          */
/* do_attend = 0 skips O6 (routing only).                                                             */
/* ------------------------------------------------------------------------------------------------ */
int hga_oracle_slice(const hga_oracle_params* p, const float* q_raw, const float* k_raw, const float* v,
                     const int* blocks, int n_blocks, int do_attend, double* k_rot_io, double* chunk_sum,
                     double* group_sum, double* q_pooled, int* chunk_idx, double* chunk_score,
                     int* n_chunks, double* chunk_all_scores, int* group_idx, double* group_score,
                     int* n_groups, double* group_cand_scores, double* out, double* lse) {
  const int G = p->G, N = p->N, D = p->D, C = p->C, gs = p->gs;
  if (G <= 0 || N <= 0 || D <= 0 || (D & 1) || C <= 0 || gs <= 0 || C % gs || N % C || p->F < 0 || p->L < 0 ||
      p->Kc < 0 || p->Kg < 0)
    return HGA_ORACLE_ERR_ARG; /* R12: only closed chunks exist -> N % C == 0 */
  const int n_b = N / C, n_g = N / gs, gpc = C / gs;
  for (size_t i = 0; i < (size_t)G * N * D; ++i)
    if (!isfinite(q_raw[i])) return HGA_ORACLE_ERR_NONFINITE; /* R8: non-finite inputs rejected */
  for (size_t i = 0; i < (size_t)N * D; ++i)
    if (!isfinite(k_raw[i]) || !isfinite(v[i])) return HGA_ORACLE_ERR_NONFINITE;

  int rc = HGA_ORACLE_OK;
  /* O1 keys */
  double* k_rot = (double*)malloc(sizeof(double) * (size_t)N * D);
  rc |= hga_oracle_rope_mod(k_raw, N, D, p->pos0, p->pos_mod, p->base, k_rot);
  /* O2 summaries from the RAW keys (the rule itself rotates), before any storage rounding (R7) */
  double* S_c = (double*)malloc(sizeof(double) * (size_t)n_b * D);
  double* S_g = (double*)malloc(sizeof(double) * (size_t)n_g * D);
  rc |= hga_oracle_summaries_mod(k_raw, N, D, C, p->n_hi_chunk, p->pos0, p->pos_mod, p->base, S_c);
  rc |= hga_oracle_summaries_mod(k_raw, N, D, gs, p->n_hi_group, p->pos0, p->pos_mod, p->base, S_g);
  /* storage rounding of K_rot for O6 (R7) */
  hga_oracle_round_io(k_rot, (size_t)N * D, p->io_bf16);
  double* vd = (double*)malloc(sizeof(double) * (size_t)N * D);
  for (size_t i = 0; i < (size_t)N * D; ++i) vd[i] = (double)v[i];
  if (k_rot_io) memcpy(k_rot_io, k_rot, sizeof(double) * (size_t)N * D);
  if (chunk_sum) memcpy(chunk_sum, S_c, sizeof(double) * (size_t)n_b * D);
  if (group_sum) memcpy(group_sum, S_g, sizeof(double) * (size_t)n_g * D);
  if (rc) goto done;

#pragma omp parallel for schedule(dynamic, 1)
  for (int bi = 0; bi < n_blocks; ++bi) {
    int j = blocks ? blocks[bi] : bi;
    if (j < 0 || j >= n_b) {
#pragma omp atomic write
      rc = HGA_ORACLE_ERR_ARG;
      continue;
    }
    /* O1 queries of block j: q_blk [G,C,D] */
    double* q_blk = (double*)malloc(sizeof(double) * (size_t)G * C * D);
    for (int h = 0; h < G; ++h)
      hga_oracle_rope_mod(q_raw + ((size_t)h * N + (size_t)j * C) * D, C, D, p->pos0 + (int64_t)j * C, p->pos_mod,
                          p->base, q_blk + (size_t)h * C * D);
    /* O3 pooled query from the un-rounded rotated queries (R7) */
    double* qbar = (double*)malloc(sizeof(double) * (size_t)D);
    hga_oracle_pool_queries(q_blk, G, C, D, C, qbar); /* a [G,C,D] tensor is one block of length C */
    if (q_pooled) memcpy(q_pooled + (size_t)bi * D, qbar, sizeof(double) * (size_t)D);
    /* O4, O5 */
    int* cidx = (int*)malloc(sizeof(int) * (size_t)(p->Kc > 0 ? p->Kc : 1));
    int* gidx = (int*)malloc(sizeof(int) * (size_t)(p->Kg > 0 ? p->Kg : 1));
    int nc, ng;
    if (group_cand_scores)
      for (int s = 0; s < p->Kc * gpc; ++s) group_cand_scores[(size_t)bi * p->Kc * gpc + s] = NAN;
    if (p->route_max) {
      /* N3 / R19: per-query scores from the rotated queries as stored */
      hga_oracle_round_io(q_blk, (size_t)G * C * D, p->io_bf16);
      nc = hga_oracle_route_chunks_max(q_blk, G * C, S_c, n_b, D, j, p->F, p->L, p->Kc, cidx,
                                       chunk_score ? chunk_score + (size_t)bi * p->Kc : NULL,
                                       chunk_all_scores ? chunk_all_scores + (size_t)bi * n_b : NULL);
      ng = hga_oracle_route_groups_max(q_blk, G * C, S_g, D, gpc, cidx, nc, p->Kg, gidx,
                                       group_score ? group_score + (size_t)bi * p->Kg : NULL,
                                       group_cand_scores ? group_cand_scores + (size_t)bi * p->Kc * gpc : NULL);
    } else {
      nc = hga_oracle_route_chunks(qbar, S_c, n_b, D, j, p->F, p->L, p->Kc, cidx,
                                   chunk_score ? chunk_score + (size_t)bi * p->Kc : NULL,
                                   chunk_all_scores ? chunk_all_scores + (size_t)bi * n_b : NULL);
      ng = hga_oracle_route_groups(qbar, S_g, D, gpc, cidx, nc, p->Kg, gidx,
                                   group_score ? group_score + (size_t)bi * p->Kg : NULL,
                                   group_cand_scores ? group_cand_scores + (size_t)bi * p->Kc * gpc : NULL);
    }
    if (chunk_idx) memcpy(chunk_idx + (size_t)bi * p->Kc, cidx, sizeof(int) * (size_t)p->Kc);
    if (group_idx) memcpy(group_idx + (size_t)bi * p->Kg, gidx, sizeof(int) * (size_t)p->Kg);
    if (n_chunks) n_chunks[bi] = nc;
    if (n_groups) n_groups[bi] = ng;
    /* O6 */
    if (do_attend && out) {
      hga_oracle_round_io(q_blk, (size_t)G * C * D, p->io_bf16);
      int r = hga_oracle_attend_block(q_blk, k_rot, vd, G, N, D, C, gs, p->F, p->L, j, gidx, p->Kg, p->scale,
                                      out + (size_t)bi * G * C * D, lse ? lse + (size_t)bi * G * C : NULL, NULL);
      if (r) {
#pragma omp atomic write
        rc = r;
      }
    }
    free(q_blk);
    free(qbar);
    free(cidx);
    free(gidx);
  }
done:
  free(k_rot);
  free(S_c);
  free(S_g);
  free(vd);
  return rc;
}

/* ------------------------------------------------------------------------------------------------ */
/* N1  One STREAMING STEP (chunk-by-chunk prefill, single-token decode, ragged prompt tail): the      */
/*     store/router cycle of PAPER.md:158 -- "appending a newly closed chunk, reading chunk summaries  */
/*     for routing, fetching group summaries for the second routing level, and gathering exact token   */
/*     K/V" -- for the token window [t0, t1) of the active chunk j = t0 / C, t1 <= (j+1) C.             */
/*     "Vectorized prefill and chunk-by-chunk decode must agree" (Table 7 :291-292).      */
/*  The function is handed ONLY the history a step may see, so causality is structural:                */
/*     q_win [G, W, D] raw queries of the window (W = t1 - t0);  k_raw, v [t1, D]: tokens 0 .. t1-1.    */
/*  Reading R17: the routing query of a step is the mean of the rotated queries of the     */
/*  rows processed in that step over the G heads (O3 restricted to the window): a whole block gives    */
/*  exactly O3; a single decode token routes with its own GQA-pooled query.                            */
/*  Order: O1 (keys 0..t1-1, window queries) -> O2 for the CLOSED chunks c < j only       */
/*  -> O3 over the window -> O4, O5 with block index j -> O6 for the window's rows.                     */
/*  Outputs (each may be NULL): q_pooled [D]; chunk_idx/score [Kc], n_chunks[1]; group_idx/score [Kg],  */
/*  n_groups[1]; out [G,W,D]; lse [G,W].                                                               */
/* ------------------------------------------------------------------------------------------------ */
int hga_oracle_step(const hga_oracle_params* p, const float* q_win, const float* k_raw, const float* v,
                    int64_t t0, int64_t t1, double* q_pooled, int* chunk_idx, double* chunk_score,
                    int* n_chunks, int* group_idx, double* group_score, int* n_groups, double* out, double* lse) {
  const int G = p->G, D = p->D, C = p->C, gs = p->gs;
  if (G <= 0 || D <= 0 || (D & 1) || C <= 0 || gs <= 0 || C % gs || p->F < 0 || p->L < 0 || p->Kc < 0 || p->Kg < 0)
    return HGA_ORACLE_ERR_ARG;
  if (t0 < 0 || t1 <= t0) return HGA_ORACLE_ERR_ARG;
  const int j = (int)(t0 / C), W = (int)(t1 - t0), r0 = (int)(t0 - (int64_t)j * C);
  if (t1 > (int64_t)(j + 1) * C) return HGA_ORACLE_ERR_ARG; /* a step stays inside the active chunk */
  const int n_hist = (int)t1, n_closed = j, gpc = C / gs;
  for (size_t i = 0; i < (size_t)G * W * D; ++i)
    if (!isfinite(q_win[i])) return HGA_ORACLE_ERR_NONFINITE;
  for (size_t i = 0; i < (size_t)n_hist * D; ++i)
    if (!isfinite(k_raw[i]) || !isfinite(v[i])) return HGA_ORACLE_ERR_NONFINITE;
  int rc = HGA_ORACLE_OK;
  double* k_rot = (double*)malloc(sizeof(double) * (size_t)n_hist * D);
  double* vd = (double*)malloc(sizeof(double) * (size_t)n_hist * D);
  double* S_c = (double*)malloc(sizeof(double) * (size_t)(n_closed > 0 ? n_closed : 1) * D);
  double* S_g = (double*)malloc(sizeof(double) * (size_t)(n_closed > 0 ? n_closed * gpc : 1) * D);
  double* q_rot = (double*)malloc(sizeof(double) * (size_t)G * W * D);
  double* qbar = (double*)malloc(sizeof(double) * (size_t)D);
  int* cidx = (int*)malloc(sizeof(int) * (size_t)(p->Kc > 0 ? p->Kc : 1));
  int* gidx = (int*)malloc(sizeof(int) * (size_t)(p->Kg > 0 ? p->Kg : 1));
  /* O1 keys of the visible history, O2 summaries of the closed chunks (from RAW keys, R7) */
  rc |= hga_oracle_rope_mod(k_raw, n_hist, D, p->pos0, p->pos_mod, p->base, k_rot);
  if (n_closed > 0) {
    rc |= hga_oracle_summaries_mod(k_raw, n_closed * C, D, C, p->n_hi_chunk, p->pos0, p->pos_mod, p->base, S_c);
    rc |= hga_oracle_summaries_mod(k_raw, n_closed * C, D, gs, p->n_hi_group, p->pos0, p->pos_mod, p->base, S_g);
  }
  hga_oracle_round_io(k_rot, (size_t)n_hist * D, p->io_bf16);
  for (size_t i = 0; i < (size_t)n_hist * D; ++i) vd[i] = (double)v[i];
  /* O1 window queries, O3 over the window (R17) */
  for (int h = 0; h < G; ++h)
    rc |= hga_oracle_rope_mod(q_win + (size_t)h * W * D, W, D, p->pos0 + t0, p->pos_mod, p->base,
                              q_rot + (size_t)h * W * D);
  rc |= hga_oracle_pool_queries(q_rot, G, W, D, W, qbar); /* a [G,W,D] tensor is one block of length W */
  if (rc) goto done;
  if (q_pooled) memcpy(q_pooled, qbar, sizeof(double) * (size_t)D);
  {
    /* O4, O5 over the closed chunks */
    int nc, ng;
    if (p->route_max) { /* N3 / R19 (with R17: the rows the step processes) */
      hga_oracle_round_io(q_rot, (size_t)G * W * D, p->io_bf16);
      nc = hga_oracle_route_chunks_max(q_rot, G * W, S_c, n_closed, D, j, p->F, p->L, p->Kc, cidx, chunk_score, NULL);
      ng = hga_oracle_route_groups_max(q_rot, G * W, S_g, D, gpc, cidx, nc, p->Kg, gidx, group_score, NULL);
    } else {
      nc = hga_oracle_route_chunks(qbar, S_c, n_closed, D, j, p->F, p->L, p->Kc, cidx, chunk_score, NULL);
      ng = hga_oracle_route_groups(qbar, S_g, D, gpc, cidx, nc, p->Kg, gidx, group_score, NULL);
    }
    if (chunk_idx) memcpy(chunk_idx, cidx, sizeof(int) * (size_t)p->Kc);
    if (group_idx) memcpy(group_idx, gidx, sizeof(int) * (size_t)p->Kg);
    if (n_chunks) *n_chunks = nc;
    if (n_groups) *n_groups = ng;
  }
  /* O6 for the window's rows */
  if (out) {
    hga_oracle_round_io(q_rot, (size_t)G * W * D, p->io_bf16);
    rc = hga_oracle_attend_rows(q_rot, k_rot, vd, G, n_hist, D, C, gs, p->F, p->L, j, r0, W, gidx, p->Kg, p->scale,
                                out, lse, NULL);
  }
done:
  free(k_rot); free(vd); free(S_c); free(S_g); free(q_rot); free(qbar); free(cidx); free(gidx);
  return rc;
}
