/*
 * foremoe_oracle.c -- plain, slow, single-threaded CPU restatement of the ForeMoE micro-step
 * plan + dispatch + combine path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or helper with the CUDA path
 * (paper_2606_11867_b200/csrc); the product never routes through it.
 *
 * Every function is the definition written out (histogram, stable counting sort, row copy,
 * weighted sum) or, for the Stage-4 token assignment the paper only sketches, the algorithm step
 * by step in the paper's order: "assign each token unit to the replica whose rank has the
 * smallest accumulated load" (Alg. 3 lines 18-21; App. D),
 * iterated "until the replicas' ranks converge toward equal utilization", with the
 * readings of DESIGN.md section 3 where the paper is silent.  No blocking, fusion or closed forms.
 *
 * Notation (Table 1): E experts, P ranks, Ns = Nb + Nr slots per rank,
 * S = P*Ns global slots, slot j belongs to rank j / Ns, K = top-k, T tokens in the step,
 * micro-step i = tokens [mb_off[i], mb_off[i+1]), instance = one (micro-step, layer),
 * pair = one (token, k) entry, c[e] = w_{s,e} with the single source rank.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   O1 hist      numpy.bincount; sums = T_i*K; closed form on constructed ids.
 *   O2 quota     brute force over ALL integer splits on tiny inputs (max rank load is the
 *                exhaustive optimum); subset closed form; ceil(LP*) of Eq.(10) by HiGHS
 *                (PAPER.md:397-407); Eq.(8)/(9) invariants; hand-worked vectors in tests/golden/.
 *                The CHOICE among optimal splits (who gets remainders) is fixed only by this
 *                file's tie-breaks: parity unpinned against the paper for that choice.
 *   O3/O4 assign numpy.argsort(kind="stable"); bijection; per-slot counts equal quotas.
 *   O5 gather    numpy fancy indexing.
 *   O6 combine   float64 sum within the fp32 error bound; exact cases (w=1, w=1/K).
 *   O7/O8 placement (Stage 1 LPT, Alg. 3 Stages 2-3): hand-worked vectors, closed forms, greedy
 *                invariants replayed in Python, structure.  O9/O10 backward: torch.autograd,
 *                adjoint identities, bf16 rounding cases (see the blocks further down).
 *   O15 (Eq.(10) with the C* term as a threshold ladder) and O16 (Alg. 2 Stage 3, replica search)
 *                restate READINGS of passages the paper leaves open: parity
 *                unpinned against the paper for the reading itself; pinned are bounds (LP, brute
 *                force), special cases, invariants and hand-worked vectors -- see their blocks.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_BAD_ARG (-1)
#define ORACLE_NO_MEM (-4)

/* data-dependent fault bits (same meaning as the library's dev_status, include/foremoe.h) */
#define FAULT_ID_RANGE 1      /* expert id outside [0, E)                          */
#define FAULT_NO_HOST 2       /* expert with tokens but no slot: Eq.(7) violated   */
#define FAULT_SLOT_EXPERT 4   /* slot_expert value outside [-1, E)                 */
#define FAULT_MB_OFF 8        /* mb_off not non-decreasing / not 0..T              */
#define FAULT_QUOTA_IN 16     /* caller quota violates Eq.(8)/(9) or is negative   */

/* ------------------------------------------------------------------------------------------
 * O1: load histogram.  hist[i][l][e] = #{(t,k): mb_off[i] <= t < mb_off[i+1], ids[l][t][k]==e}
 * (w_{s,e} of PAPER.md:204/:247 with one source); step_hist[l][e] = sum_i hist[i][l][e]
 * (the aggregate of PAPER.md:284).  Returns fault bits.
 * ------------------------------------------------------------------------------------------ */
int oracle_load_hist(int L, int T, int K, int E, int n_mb, const int32_t *ids,
                     const int32_t *mb_off, int32_t *hist, int64_t *step_hist) {
  int fault = 0;
  memset(hist, 0, sizeof(int32_t) * (size_t)n_mb * L * E);
  if (step_hist) memset(step_hist, 0, sizeof(int64_t) * (size_t)L * E);
  if (mb_off[0] != 0 || mb_off[n_mb] != T) fault |= FAULT_MB_OFF;
  for (int i = 0; i < n_mb; i++)
    if (mb_off[i + 1] < mb_off[i]) fault |= FAULT_MB_OFF;
  if (fault) return fault;
  for (int i = 0; i < n_mb; i++)
    for (int l = 0; l < L; l++)
      for (int t = mb_off[i]; t < mb_off[i + 1]; t++)
        for (int k = 0; k < K; k++) {
          int32_t e = ids[((size_t)l * T + t) * K + k];
          if (e < 0 || e >= E) { fault |= FAULT_ID_RANGE; continue; }
          hist[((size_t)i * L + l) * E + e] += 1;
          if (step_hist) step_hist[(size_t)l * E + e] += 1;
        }
  return fault;
}

/* ------------------------------------------------------------------------------------------
 * O2: Stage-4 token assignment as integer quotas for ONE instance.
 *
 * c[E] counts, slot_expert[S] placement (-1 = empty slot).  Outputs quota[S], rank_load[P],
 * slot_off[S+1].  stop_after: 1 = Phase A + ONE water-filling pass (the literal single pass of
 * Alg. 3 lines 18-21), 2 = Phase B fixpoint, 3 = Phase C too (the rule).  stats[0] = passes run,
 * stats[1] = units moved by Phase C.  Returns fault bits.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
  int E, P, Ns, S;
  const int32_t *c;
  const int32_t *slot_expert;
  int32_t *active;    /* [S] 1 if slot is the lowest-indexed slot of its expert on its rank */
  int32_t *n_active;  /* [E] number of active hosts */
  int32_t *host_ptr;  /* [E+1] active hosts of e = host_slot[host_ptr[e] .. host_ptr[e+1]) */
  int32_t *host_slot; /* [S]   ... in ascending slot index */
  int64_t *load;      /* [P] */
  int32_t *q;         /* [S] */
} inst_t;

/* a before b in the processing order: descending count, ties ascending expert id (reading 3) */
static int goes_before(const int32_t *c, int32_t ea, int32_t eb) {
  if (c[ea] != c[eb]) return c[ea] > c[eb];
  return ea < eb;
}

/* water-fill one replicated expert, unit by unit: each unit goes to the active
 * host whose rank currently has the smallest load, ties to the lowest slot index. */
static void fill_units(inst_t *I, int e) {
  for (int32_t u = 0; u < I->c[e]; u++) {
    int best = -1;
    for (int a = I->host_ptr[e]; a < I->host_ptr[e + 1]; a++) {   /* ascending slot index */
      int j = I->host_slot[a];
      if (best < 0 || I->load[j / I->Ns] < I->load[best / I->Ns]) best = j;
    }
    I->q[best] += 1;
    I->load[best / I->Ns] += 1;
  }
}

int oracle_quota(int E, int P, int Ns, const int32_t *c, const int32_t *slot_expert,
                 int32_t *quota, int32_t *rank_load, int32_t *slot_off, int stop_after,
                 int32_t *stats) {
  const int S = P * Ns;
  int fault = 0;
  inst_t I;
  I.E = E; I.P = P; I.Ns = Ns; I.S = S; I.c = c; I.slot_expert = slot_expert;
  I.active = (int32_t *)calloc((size_t)S, sizeof(int32_t));
  I.n_active = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  I.load = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  I.q = (int32_t *)calloc((size_t)S, sizeof(int32_t));
  I.host_ptr = (int32_t *)calloc((size_t)E + 1, sizeof(int32_t));
  I.host_slot = (int32_t *)calloc((size_t)S + 1, sizeof(int32_t));
  int32_t *R = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *old = (int32_t *)calloc((size_t)S, sizeof(int32_t));
  int32_t *visited = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int32_t *par_rank = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int32_t *par_exp = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int32_t *queue = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  if (stats) { stats[0] = 0; stats[1] = 0; }
  if (!I.host_ptr || !I.host_slot || !I.active || !I.n_active || !I.load || !I.q || !R || !old || !visited || !par_rank ||
      !par_exp || !queue) { fault = ORACLE_NO_MEM; goto done; }

  /* hosts: active = lowest-indexed slot of expert e on its rank (reading 10) */
  for (int j = 0; j < S; j++) {
    int32_t e = slot_expert[j];
    if (e < -1 || e >= E) { fault |= FAULT_SLOT_EXPERT; continue; }
    if (e < 0) continue;
    int first = 1;
    for (int j2 = (j / Ns) * Ns; j2 < j; j2++)
      if (slot_expert[j2] == e) first = 0;
    I.active[j] = first;
    I.n_active[e] += first;
  }
  for (int e = 0; e < E; e++) {          /* active host lists, ascending slot index */
    I.host_ptr[e + 1] = I.host_ptr[e];
    for (int j = 0; j < S; j++)
      if (slot_expert[j] == e && I.active[j]) I.host_slot[I.host_ptr[e + 1]++] = j;
  }
  for (int e = 0; e < E; e++) {
    if (c[e] < 0) fault |= FAULT_ID_RANGE;
    if (c[e] > 0 && I.n_active[e] == 0) fault |= FAULT_NO_HOST;
  }
  if (fault) goto write_out;

  /* Phase A: forced load of singly hosted experts */
  int nR = 0;
  for (int e = 0; e < E; e++) {
    if (I.n_active[e] == 1) {
      for (int j = 0; j < S; j++)
        if (slot_expert[j] == e && I.active[j]) { I.q[j] = c[e]; I.load[j / Ns] += c[e]; }
    } else if (I.n_active[e] >= 2) {
      R[nR++] = e;
    }
  }
  /* replicated experts in descending count, ties ascending id (reading 3) */
  for (int a = 1; a < nR; a++) {          /* insertion sort */
    int32_t e = R[a];
    int b = a;
    while (b > 0 && goes_before(c, e, R[b - 1])) { R[b] = R[b - 1]; b--; }
    R[b] = e;
  }

  /* Phase B: Gauss-Seidel water-filling passes until a full pass changes no quota (cap 256) */
  int passes = 0;
  for (int pass = 0; pass < 256; pass++) {
    int changed = 0;
    passes++;
    for (int a = 0; a < nR; a++) {
      int e = R[a];
      for (int j = 0; j < S; j++)
        if (slot_expert[j] == e && I.active[j]) {
          old[j] = I.q[j];
          I.load[j / Ns] -= I.q[j];
          I.q[j] = 0;
        }
      fill_units(&I, e);
      for (int j = 0; j < S; j++)
        if (slot_expert[j] == e && I.active[j] && I.q[j] != old[j]) changed = 1;
    }
    if (!changed || stop_after == 1) break;
  }
  if (stats) stats[0] = passes;

  /* Phase C: unit augmentations until the lowest max-load rank has no improving path */
  if (stop_after >= 3) {
    for (;;) {
      int64_t mx = -1; int h = 0;
      for (int r = 0; r < P; r++) if (I.load[r] > mx) { mx = I.load[r]; h = r; }
      memset(visited, 0, sizeof(int32_t) * (size_t)P);
      int head = 0, tail = 0, target = -1;
      visited[h] = 1; queue[tail++] = h; par_rank[h] = -1; par_exp[h] = -1;
      while (head < tail && target < 0) {
        int r = queue[head++];
        /* replicated experts with quota on r, ascending expert id */
        for (int e = 0; e < E && target < 0; e++) {
          if (I.n_active[e] < 2) continue;
          int on_r = -1;
          for (int j = r * Ns; j < (r + 1) * Ns; j++)
            if (slot_expert[j] == e && I.active[j]) on_r = j;
          if (on_r < 0 || I.q[on_r] <= 0) continue;
          for (int j = 0; j < S && target < 0; j++) {   /* active hosts, ascending slot index */
            if (slot_expert[j] != e || !I.active[j]) continue;
            int r2 = j / Ns;
            if (visited[r2]) continue;
            visited[r2] = 1; par_rank[r2] = r; par_exp[r2] = e; queue[tail++] = r2;
            if (I.load[r2] <= mx - 2) target = r2;
          }
        }
      }
      if (target < 0) break;
      /* move one unit of each expert on the path target <- ... <- h */
      for (int r2 = target; par_rank[r2] >= 0; r2 = par_rank[r2]) {
        int r = par_rank[r2], e = par_exp[r2];
        for (int j = r * Ns; j < (r + 1) * Ns; j++)
          if (slot_expert[j] == e && I.active[j]) I.q[j] -= 1;
        for (int j = r2 * Ns; j < (r2 + 1) * Ns; j++)
          if (slot_expert[j] == e && I.active[j]) I.q[j] += 1;
      }
      I.load[h] -= 1;
      I.load[target] += 1;
      if (stats) stats[1] += 1;
    }
  }

write_out:
  slot_off[0] = 0;
  for (int j = 0; j < S; j++) {
    quota[j] = I.q[j];
    slot_off[j + 1] = slot_off[j] + I.q[j];
  }
  for (int r = 0; r < P; r++) {
    int64_t s = 0;
    for (int j = r * Ns; j < (r + 1) * Ns; j++) s += I.q[j];
    rank_load[r] = (int32_t)s;
  }
done:
  free(I.host_ptr); free(I.host_slot); free(I.active); free(I.n_active); free(I.load); free(I.q); free(R); free(old);
  free(visited); free(par_rank); free(par_exp); free(queue);
  return fault;
}

/* validate a caller-supplied quota against Eq.(8) conservation and Eq.(9) feasibility
 * (PAPER.md:266-270): sum over hosts of e equals c[e]; quota > 0 only on slots holding e. */
int oracle_check_quota(int E, int S, const int32_t *c, const int32_t *slot_expert,
                       const int32_t *quota) {
  int fault = 0;
  int64_t *sum = (int64_t *)calloc((size_t)E, sizeof(int64_t));
  if (!sum) return ORACLE_NO_MEM;
  for (int j = 0; j < S; j++) {
    if (quota[j] < 0) fault |= FAULT_QUOTA_IN;
    if (slot_expert[j] < 0) { if (quota[j] != 0) fault |= FAULT_QUOTA_IN; continue; }
    sum[slot_expert[j]] += quota[j];
  }
  for (int e = 0; e < E; e++) if (sum[e] != c[e]) fault |= FAULT_QUOTA_IN;
  free(sum);
  return fault;
}

/* ------------------------------------------------------------------------------------------
 * O3 + O4 for ONE instance: n_pairs = T_i*K ids in (t,k) order.
 * O3: the pair with 0-based rank n among the instance's pairs of expert e goes to the host slot
 *     j of e (ascending slot index) whose cumulative-quota interval contains n (reading 1:
 *     contiguous blocks of the expert's stable token order; PAPER.md:250 gives only fractions).
 * O4: stable counting sort by slot: dst = slot_off[j] + #{earlier pairs with slot j};
 *     inv[p] = base + dst, perm[base + dst] = base + p, where base = mb_off[i]*K places the
 *     instance's rows inside its layer (layer-global row indices).
 * ------------------------------------------------------------------------------------------ */
int oracle_assign_instance(int E, int S, int n_pairs, int32_t base, const int32_t *ids,
                           const int32_t *slot_expert, const int32_t *quota,
                           const int32_t *slot_off, int32_t *pair_slot, int32_t *inv,
                           int32_t *perm) {
  int fault = 0;
  int32_t *seen = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *filled = (int32_t *)calloc((size_t)S, sizeof(int32_t));
  if (!seen || !filled) { free(seen); free(filled); return ORACLE_NO_MEM; }
  for (int p = 0; p < n_pairs; p++) {
    int32_t e = ids[p];
    if (e < 0 || e >= E) { fault |= FAULT_ID_RANGE; pair_slot[p] = -1; continue; }
    int32_t n = seen[e]++;
    int32_t cum = 0, slot = -1;
    for (int j = 0; j < S; j++) {
      if (slot_expert[j] != e) continue;
      if (n < cum + quota[j]) { slot = j; break; }
      cum += quota[j];
    }
    pair_slot[p] = slot;
    if (slot < 0) fault |= FAULT_NO_HOST;
  }
  for (int p = 0; p < n_pairs; p++) {
    int32_t j = pair_slot[p];
    if (j < 0) { inv[p] = -1; continue; }
    int32_t dst = slot_off[j] + filled[j]++;
    inv[p] = base + dst;
    perm[dst] = base + p;
  }
  free(seen); free(filled);
  return fault;
}

/* ------------------------------------------------------------------------------------------
 * O5: gather (dispatch).  buf[d][:] = x[(perm[d] - pair_base) / K][:], bit copy of row_bytes.
 * perm holds n_rows layer-global pair indices; pair_base = first token of the range * K; x row 0
 * is that first token; buf row 0 is layer-global row pair_base.  (dispatch "routes
 * each token ... to the rank hosting its assigned expert".)
 * ------------------------------------------------------------------------------------------ */
int oracle_gather(int64_t n_rows, int K, int64_t row_bytes, int32_t pair_base,
                  const int32_t *perm, const uint8_t *x, uint8_t *buf) {
  for (int64_t d = 0; d < n_rows; d++) {
    int64_t t = ((int64_t)perm[d] - pair_base) / K;
    memcpy(buf + d * row_bytes, x + t * row_bytes, (size_t)row_bytes);
  }
  return 0;
}

static float bf16_to_float(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  memcpy(&f, &u, sizeof f);
  return f;
}

/* ------------------------------------------------------------------------------------------
 * O6: combine.  y[t][h] = sum_{k=0}^{K-1} w[t][k] * float(eo[inv[t*K+k] - row_base][h]),
 * accumulated as acc = fmaf(w, v, acc) from acc = 0.0f with k ascending, fp32 output
 * ("the weighted sum of the selected experts' outputs, where the weights are the
 * corresponding router probabilities"; order / fma / output type = reading 16).
 * act_dtype 0 = bf16 rows, 1 = fp32 rows.  A pair with inv < 0 (faulted in the plan: its expert id
 * was out of range or had no host) has no dispatched row: it is skipped, like in O9 / O10
 * (include/foremoe.h: "pairs with inv < 0 contribute nothing"; reading 38).
 * ------------------------------------------------------------------------------------------ */
int oracle_combine(int64_t n_tok, int K, int H, int act_dtype, int32_t row_base,
                   const int32_t *inv, const float *w, const void *eo, float *y) {
  for (int64_t t = 0; t < n_tok; t++)
    for (int h = 0; h < H; h++) {
      float acc = 0.0f;
      for (int k = 0; k < K; k++) {
        if (inv[t * K + k] < 0) continue;      /* faulted pair: contributes nothing (as O9 / O10) */
        int64_t row = (int64_t)inv[t * K + k] - row_base;
        float v = act_dtype == 0 ? bf16_to_float(((const uint16_t *)eo)[row * H + h])
                                 : ((const float *)eo)[row * H + h];
        acc = fmaf(w[t * K + k], v, acc);
      }
      y[t * H + h] = acc;
    }
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * Whole-step plan: O1 must have been run (hist).  For every instance (i,l): O2 then O3+O4.
 * quota_in (may be NULL): caller-supplied quotas, validated by Eq.(8)/(9) instead of computed.
 * ------------------------------------------------------------------------------------------ */
int oracle_plan(int L, int T, int K, int E, int P, int Ns, int n_mb, const int32_t *ids,
                const int32_t *mb_off, const int32_t *hist, const int32_t *slot_expert,
                const int32_t *quota_in, int32_t *quota, int32_t *rank_load, int32_t *slot_off,
                int32_t *pair_slot, int32_t *inv, int32_t *perm) {
  const int S = P * Ns;
  int fault = 0;
  for (int i = 0; i < n_mb; i++)
    for (int l = 0; l < L; l++) {
      size_t inst = (size_t)i * L + l;
      const int32_t *c = hist + inst * E;
      const int32_t *se = slot_expert + (size_t)l * S;
      int32_t *q = quota + inst * S, *so = slot_off + inst * (S + 1);
      if (quota_in) {
        fault |= oracle_check_quota(E, S, c, se, quota_in + inst * S);
        so[0] = 0;
        for (int j = 0; j < S; j++) { q[j] = quota_in[inst * S + j]; so[j + 1] = so[j] + q[j]; }
        for (int r = 0; r < P; r++) {
          int32_t s = 0;
          for (int j = r * Ns; j < (r + 1) * Ns; j++) s += q[j];
          rank_load[inst * P + r] = s;
        }
      } else {
        fault |= oracle_quota(E, P, Ns, c, se, q, rank_load + inst * P, so, 3, NULL);
      }
      if (fault & (FAULT_NO_HOST | FAULT_SLOT_EXPERT | FAULT_QUOTA_IN)) continue;
      size_t p0 = ((size_t)l * T + mb_off[i]) * K;
      int n_pairs = (mb_off[i + 1] - mb_off[i]) * K;
      fault |= oracle_assign_instance(E, S, n_pairs, mb_off[i] * K, ids + p0, se, q, so,
                                      pair_slot + p0, inv + p0, perm + p0);
    }
  return fault;
}

/* ==========================================================================================
 * NEXT row: placements computed from the foresight.
 *
 * O7 oracle_base_placement: Stage 1 at rank level (Alg. 1 lines 13-21, prose
 *   :290): experts in descending aggregate load, each to the currently least-loaded rank ("LPT").
 *   The output "fills the N_b base slots on every rank", so a rank is eligible only
 *   while it has a free base slot (the listing omits this capacity; reading 21).
 *   One machine (M = 1): the machine-level greedy of Alg. 1 lines 5-12 needs per-source loads and
 *   the time-model coefficients K1, K2 the paper never gives -- out of scope.
 *
 * O8 oracle_microstep_placement: Alg. 3 Stages 2-3 (prose :840-842) for ONE
 *   (micro-step, layer) instance, machines = M groups of R = P / M consecutive ranks; an expert
 *   is local to the machine of its base rank.
 *   Stage 2 (lines 4-10): local experts in descending micro-step load, each to the least-loaded
 *     local rank with a free base slot; RL[r] += load.
 *   Stage 3 (lines 12-16): R * N_r rounds per machine: e* = the locally heaviest expert, r* = the
 *     local rank with the minimum current load; place a replica of e* on r* and update RL.
 *   Readings: "heaviest" = largest load per copy c[e] / copies[e] (compared
 *   exactly by cross-multiplication), ties lower id, among experts that still have an eligible
 *   rank (free redundant slot, not hosting e* yet); an expert whose per-copy load is 0 is never
 *   replicated (remaining slots stay empty, -1); "update RL" = every host of e* carries the exact
 *   integer even split floor(c/n) (+1 for the first c mod n hosts in ascending slot index);
 *   all ties between ranks go to the lowest rank.
 * Both return fault bits (FAULT_SLOT_EXPERT: base placement unusable; FAULT_ID_RANGE: negative load).
 * ========================================================================================== */
static int heavier(const int64_t *c, int a, int b) {   /* a before b: descending load, ties ascending id */
  if (c[a] != c[b]) return c[a] > c[b];
  return a < b;
}

int oracle_base_placement(int E, int P, int Nb, int Nr, const int64_t *tot, int32_t *slot_expert) {
  const int Ns = Nb + Nr, S = P * Ns;
  int fault = 0;
  for (int j = 0; j < S; j++) slot_expert[j] = -1;
  if ((int64_t)P * Nb < E) return FAULT_SLOT_EXPERT;
  int32_t *order = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int64_t *RL = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  int32_t *nb = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  if (!order || !RL || !nb) { free(order); free(RL); free(nb); return ORACLE_NO_MEM; }
  for (int e = 0; e < E; e++) {
    if (tot[e] < 0) fault |= FAULT_ID_RANGE;
    order[e] = e;
  }
  for (int a = 1; a < E; a++) {          /* insertion sort: descending load, ties ascending id */
    int32_t e = order[a];
    int b = a;
    while (b > 0 && heavier(tot, e, order[b - 1])) { order[b] = order[b - 1]; b--; }
    order[b] = e;
  }
  for (int a = 0; a < E && !fault; a++) {
    const int e = order[a];
    int best = -1;
    for (int r = 0; r < P; r++)
      if (nb[r] < Nb && (best < 0 || RL[r] < RL[best])) best = r;   /* ties: lowest rank */
    slot_expert[best * Ns + nb[best]] = e;
    nb[best] += 1;
    RL[best] += tot[e];
  }
  free(order); free(RL); free(nb);
  return fault;
}

/* exact integer even split of c over n hosts: host idx (ascending slot order) carries this much */
static int64_t even_share(int64_t c, int n, int idx) { return c / n + (idx < c % n ? 1 : 0); }

static int microstep_impl(int E, int P, int Nb, int Nr, int M, const int32_t *c32,
                          const int32_t *base_se, int32_t *out_se, int relocate) {
  const int Ns = Nb + Nr, S = P * Ns;
  int fault = 0;
  for (int j = 0; j < S; j++) out_se[j] = -1;
  if (M <= 0 || P % M != 0) return ORACLE_BAD_ARG;
  const int R = P / M;
  int64_t *c = (int64_t *)calloc((size_t)E, sizeof(int64_t));
  int32_t *mach = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *order = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int64_t *RL = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  int32_t *nb = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int32_t *nr = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int32_t *copies = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *dead = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *hosts = (int32_t *)calloc((size_t)S + 1, sizeof(int32_t));   /* scratch: slots of e*, ascending */
  if (!c || !mach || !order || !RL || !nb || !nr || !copies || !dead || !hosts) { fault = ORACLE_NO_MEM; goto done; }

  for (int e = 0; e < E; e++) { c[e] = c32[e]; if (c32[e] < 0) fault |= FAULT_ID_RANGE; mach[e] = -1; }
  for (int j = S - 1; j >= 0; j--) {       /* machine of e = machine of its lowest-indexed base slot */
    if (!relocate && j % Ns >= Nb) continue;   /* O13 does not read the input's redundant slots */
    const int32_t e = base_se[j];
    if (e < -1 || e >= E) { fault |= FAULT_SLOT_EXPERT; continue; }
    if (e >= 0) mach[e] = (j / Ns) / R;
  }
  for (int m = 0; m < M; m++) {
    int n_local = 0;
    for (int e = 0; e < E; e++) n_local += (mach[e] == m);
    if (n_local > R * Nb) fault |= FAULT_SLOT_EXPERT;
  }
  for (int e = 0; e < E; e++) if (mach[e] < 0) fault |= FAULT_SLOT_EXPERT;
  if (fault) goto done;

  for (int e = 0; e < E; e++) order[e] = e;
  for (int a = 1; a < E; a++) {
    int32_t e = order[a];
    int b = a;
    while (b > 0 && heavier(c, e, order[b - 1])) { order[b] = order[b - 1]; b--; }
    order[b] = e;
  }
  if (!relocate) {
    /* O13: the relocation was done by someone else (Alg. 2 Stage 2 swaps, O12): every expert stays in
     * the base slot it was given; the input must hold each expert exactly once in the base slots */
    for (int e = 0; e < E; e++) {
      int n = 0, at = -1;
      for (int j = 0; j < S; j++)
        if (base_se[j] == e && j % Ns < Nb) { n++; if (at < 0) at = j; }
      if (n != 1) { fault |= FAULT_SLOT_EXPERT; continue; }
      out_se[at] = e;
      mach[e] = (at / Ns) / R;                 /* the input's redundant slots are ignored */
      nb[at / Ns] += 1;
      RL[at / Ns] += c[e];
      copies[e] = 1;
    }
    if (fault) { for (int j = 0; j < S; j++) out_se[j] = -1; goto done; }
  }
  /* Stage 2: LPT relocation inside each machine (Alg. 3 lines 4-10) */
  for (int a = 0; a < E && relocate; a++) {
    const int e = order[a], m = mach[e];
    int best = -1;
    for (int r = m * R; r < (m + 1) * R; r++)
      if (nb[r] < Nb && (best < 0 || RL[r] < RL[best])) best = r;
    out_se[best * Ns + nb[best]] = e;
    nb[best] += 1;
    RL[best] += c[e];
    copies[e] = 1;
  }
  /* Stage 3: replication, R * N_r rounds per machine (Alg. 3 lines 12-16) */
  for (int m = 0; m < M; m++) {
    for (int k = 0; k < R * Nr; k++) {
      int estar = -1, rstar = -1;
      for (;;) {
        estar = -1;                       /* locally heaviest per copy, ties lower id, not ruled out */
        for (int e = 0; e < E; e++) {
          if (mach[e] != m || dead[e] || c[e] <= 0) continue;
          if (estar < 0 || c[e] * copies[estar] > c[estar] * copies[e]) estar = e;
        }
        if (estar < 0) break;
        rstar = -1;                       /* least-loaded eligible local rank, ties lowest rank */
        for (int r = m * R; r < (m + 1) * R; r++) {
          if (nr[r] >= Nr) continue;
          int hosted = 0;
          for (int j = r * Ns; j < (r + 1) * Ns; j++) hosted |= (out_se[j] == estar);
          if (hosted) continue;
          if (rstar < 0 || RL[r] < RL[rstar]) rstar = r;
        }
        if (rstar >= 0) break;
        dead[estar] = 1;                  /* no eligible rank now => none later either */
      }
      if (estar < 0) break;
      /* update RL: even split over n hosts -> even split over n + 1 hosts */
      int n = 0;
      for (int j = 0; j < S; j++) if (out_se[j] == estar) hosts[n++] = j;
      for (int a = 0; a < n; a++) RL[hosts[a] / Ns] -= even_share(c[estar], n, a);
      out_se[rstar * Ns + Nb + nr[rstar]] = estar;
      nr[rstar] += 1;
      copies[estar] += 1;
      n = 0;
      for (int j = 0; j < S; j++) if (out_se[j] == estar) hosts[n++] = j;
      for (int a = 0; a < n; a++) RL[hosts[a] / Ns] += even_share(c[estar], n, a);
    }
  }
done:
  free(c); free(mach); free(order); free(RL); free(nb); free(nr); free(copies); free(dead); free(hosts);
  return fault;
}

int oracle_microstep_placement(int E, int P, int Nb, int Nr, int M, const int32_t *c32,
                               const int32_t *base_se, int32_t *out_se) {
  return microstep_impl(E, P, Nb, Nr, M, c32, base_se, out_se, 1);
}

/* O13 oracle_replication: Stage 3 alone (Alg. 3 lines 12-16 / the replication loop of Alg. 2 lines
 * 14-19 with Alg. 3's choice rule, readings 22-25) on a placement whose base slots are already
 * final -- e.g. the output of O12 -- so that swaps (Alg. 2 Stage 2) + replication + Stage 4 compose.
 * Redundant slots of the input are ignored and rebuilt.  Pins: equals O8 when fed O8's own Stage-2
 * result; structure; first replica = heaviest expert on the least-loaded other rank. */
int oracle_replication(int E, int P, int Nb, int Nr, int M, const int32_t *c32,
                       const int32_t *placed_se, int32_t *out_se) {
  return microstep_impl(E, P, Nb, Nr, M, c32, placed_se, out_se, 0);
}

/* ==========================================================================================
 * NEXT row: backward of the data path, the policy-update stage.
 * "the backward pass triggers an additional gradient computation and additional MoE dispatch and
 * MoE combine of gradients" (sec. 7.1, n1 = 3, n2 = 4); "the forward and backward
 * passes of the same micro-step use the same reconfiguration plan" (PAPER.md:170 Fig. 7, :188),
 * i.e. the SAME inv / w as the forward.  Forward: buf = gather(x) (O5), eo = expert(buf),
 * y = combine(eo, w) (O6).  Given dy = dLoss/dy (fp32, like y), the chain rule gives
 *
 * O9 oracle_combine_bwd ("MoE dispatch of gradients": token order -> slot order)
 *     d_eo[inv[t*K+k] - row_base][h] = round_act( w[t][k] * dy[t][h] )      one fp32 multiply, then
 *                                      round-to-nearest-even to bf16 when act_dtype == 0
 *     dw[t][k] = sum_h dy[t][h] * float(eo[inv[t*K+k] - row_base][h])       plain definition,
 *                                      accumulated in fp64, rounded once to fp32
 *   Readings: gradient rows have the activation dtype, the rounding decision is
 *   taken on the fp32 product (the kernel's precision); dw is defined exactly (the GPU reduces in
 *   fp32 in another order and is compared within H * 2^-24 * sum_h |dy * eo|); pairs with
 *   inv < 0 are skipped (rows untouched, dw = 0).
 *
 * O10 oracle_dispatch_bwd ("MoE combine of gradients": slot order -> token order)
 *     dx[t][h] = sum_{k=0}^{K-1} float(d_buf[inv[t*K+k] - row_base][h])     fp32 adds, k ascending
 *   from 0.0f (the transpose of the row gather: token t was copied to its K rows) -- the same
 *   fixed order as O6, which it equals with all weights 1.
 * Pins (tests/test_oracle_backward.py): torch.autograd on a float64 forward built from
 * index_select / einsum; the adjoint identities <C(eo), dy> = <eo, C^T(dy)>, <D(x), g> = <x, D^T(g)>;
 * bf16 rounding against torch's conversion and against hand-picked tie cases; closed forms.
 * ========================================================================================== */
static uint16_t float_to_bf16_rne(float f) {
  uint32_t u;
  memcpy(&u, &f, sizeof u);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x0040u);   /* NaN stays NaN (quiet) */
  uint32_t lsb = (u >> 16) & 1u;
  u += 0x7fffu + lsb;                       /* round to nearest, ties to even */
  return (uint16_t)(u >> 16);
}

int oracle_combine_bwd(int64_t n_tok, int K, int H, int act_dtype, int32_t row_base,
                       const int32_t *inv, const float *w, const float *dy,
                       const void *eo /* may be NULL with dw */, void *d_eo, float *dw /* may be NULL */) {
  for (int64_t t = 0; t < n_tok; t++)
    for (int k = 0; k < K; k++) {
      if (inv[t * K + k] < 0) { if (dw) dw[t * K + k] = 0.0f; continue; }
      int64_t row = (int64_t)inv[t * K + k] - row_base;
      double dot = 0.0;
      for (int h = 0; h < H; h++) {
        float g = w[t * K + k] * dy[t * H + h];
        if (act_dtype == 0) ((uint16_t *)d_eo)[row * H + h] = float_to_bf16_rne(g);
        else ((float *)d_eo)[row * H + h] = g;
        if (dw && eo) {
          float v = act_dtype == 0 ? bf16_to_float(((const uint16_t *)eo)[row * H + h])
                                   : ((const float *)eo)[row * H + h];
          dot += (double)dy[t * H + h] * (double)v;
        }
      }
      if (dw) dw[t * K + k] = (float)dot;
    }
  return 0;
}

int oracle_dispatch_bwd(int64_t n_tok, int K, int H, int act_dtype, int32_t row_base,
                        const int32_t *inv, const void *d_buf, float *dx) {
  for (int64_t t = 0; t < n_tok; t++)
    for (int h = 0; h < H; h++) {
      float acc = 0.0f;
      for (int k = 0; k < K; k++) {
        if (inv[t * K + k] < 0) continue;
        int64_t row = (int64_t)inv[t * K + k] - row_base;
        float v = act_dtype == 0 ? bf16_to_float(((const uint16_t *)d_buf)[row * H + h])
                                 : ((const float *)d_buf)[row * H + h];
        acc = acc + v;
      }
      dx[t * H + h] = acc;
    }
  return 0;
}

/* ==========================================================================================
 * NEXT row: per-source, multi-machine Stage 4.
 *
 * Inputs now carry the source of every token: w_{s,e} is a P x E matrix, the
 * P ranks form M machines of R = P / M consecutive ranks, and C_{i,j} of Eq.(5)
 * counts the tokens flowing from the ranks of machine i to the slots of machine j.
 *
 * O11 oracle_quota_local: token assignment with the placement fixed, by the paper's
 * "locality-aware token assignment heuristic: tokens prefer same-machine replicas to avoid
 * cross-machine traffic, and any leftover tokens are routed to minimize per-rank load"
 * (sec. 8.2), made exact in the same way as O2 (readings 29-31):
 *   - commodity (e, m) = the tokens of expert e whose source rank sits on machine m; only the
 *     machine of the source matters for L_r (Eq.(4)) and C_{i,j} (Eq.(5)), so sources are
 *     aggregated per machine: c[e][m] = sum_{s in ranks(m)} w_{s,e};
 *   - allowed hosts of (e, m): the slots holding e on machine m if there is one ("prefer
 *     same-machine replicas"), else every slot holding e ("leftover tokens");
 *   - among all integer assignments that respect the allowed hosts, minimise L_max: this is O2
 *     itself on a VIRTUAL instance with experts v = e * M + m, counts c[e][m] and virtual slots
 *     (j, m) -> index j * M + m, N_s * M per rank, holding v when slot j is an allowed host of
 *     (e, m) and -1 otherwise.  The reduction is written out below and oracle_quota (O2, pinned)
 *     is called on it, so every tie-break of O2 carries over: commodities in descending count,
 *     ties ascending v; units to the least-loaded rank, ties to the lowest virtual slot.
 * Outputs: q_src[m][j] (tokens of source machine m sent to slot j), rank_load[r],
 * traffic[i][j] = sum over slots of machine j of q_src[i][.] (diagonal = tokens that stay inside
 * the machine; off-diagonal = C_{i,j} of Eq.(5)).
 * Pins (tests/test_oracle_local.py): brute force over all integer splits within the allowed
 * hosts on tiny instances; ceil(LP*) of Eq.(10) restricted to the allowed hosts (HiGHS); total
 * cross-machine traffic equals its lower bound (tokens with no same-machine replica); M = 1 is O2;
 * experts hosted on one machine only => same max load as O2 on the summed counts; hand-worked
 * vectors in tests/golden/local_vectors.json.
 * ========================================================================================== */
int oracle_local_placement(int E, int P, int Ns, int M, const int32_t *slot_expert,
                           int32_t *slot_expert_v /* [P*Ns*M] */) {
  const int S = P * Ns;
  if (M <= 0 || P % M != 0) return ORACLE_BAD_ARG;
  const int R = P / M;
  int fault = 0;
  for (int j = 0; j < S; j++) {
    const int32_t e = slot_expert[j];
    if (e < -1 || e >= E) fault |= FAULT_SLOT_EXPERT;
    for (int m = 0; m < M; m++) {
      int32_t v = -1;
      if (e >= 0 && e < E) {
        const int mj = (j / Ns) / R;               /* machine of slot j */
        int local_exists = 0;                      /* does machine m hold e at all? */
        for (int j2 = 0; j2 < S; j2++)
          if (slot_expert[j2] == e && (j2 / Ns) / R == m) local_exists = 1;
        if (mj == m || !local_exists) v = e * M + m;
      }
      slot_expert_v[(size_t)j * M + m] = v;
    }
  }
  return fault;
}

int oracle_quota_local(int E, int P, int Ns, int M, const int32_t *w_se /* [P][E] per-source counts */,
                       const int32_t *slot_expert, int32_t *q_src /* [M][S] */,
                       int32_t *rank_load /* [P] */, int32_t *traffic /* [M][M] */,
                       int32_t *quota_v /* [S*M] or NULL */, int32_t *slot_off_v /* [S*M+1] or NULL */) {
  const int S = P * Ns;
  if (M <= 0 || P % M != 0) return ORACLE_BAD_ARG;
  const int R = P / M;
  int32_t *c_v = (int32_t *)calloc((size_t)E * M, sizeof(int32_t));
  int32_t *se_v = (int32_t *)calloc((size_t)S * M, sizeof(int32_t));
  int32_t *q_v = (int32_t *)calloc((size_t)S * M, sizeof(int32_t));
  int32_t *so_v = (int32_t *)calloc((size_t)S * M + 1, sizeof(int32_t));
  int fault;
  if (!c_v || !se_v || !q_v || !so_v) { fault = ORACLE_NO_MEM; goto done; }
  for (int s = 0; s < P; s++)                      /* aggregate the sources of a machine */
    for (int e = 0; e < E; e++) c_v[e * M + s / R] += w_se[(size_t)s * E + e];
  fault = oracle_local_placement(E, P, Ns, M, slot_expert, se_v);
  if (fault < 0) goto done;
  fault |= oracle_quota(E * M, P, Ns * M, c_v, se_v, q_v, rank_load, so_v, 3, NULL);
  if (fault < 0) goto done;
  for (int m = 0; m < M; m++)
    for (int j = 0; j < S; j++) q_src[(size_t)m * S + j] = q_v[(size_t)j * M + m];
  for (int i = 0; i < M; i++)
    for (int mj = 0; mj < M; mj++) {
      int64_t t = 0;
      for (int j = mj * R * Ns; j < (mj + 1) * R * Ns; j++) t += q_src[(size_t)i * S + j];
      traffic[i * M + mj] = (int32_t)t;
    }
  if (quota_v) memcpy(quota_v, q_v, sizeof(int32_t) * (size_t)S * M);
  if (slot_off_v) memcpy(slot_off_v, so_v, sizeof(int32_t) * ((size_t)S * M + 1));
done:
  free(c_v); free(se_v); free(q_v); free(so_v);
  return fault;
}

/* ==========================================================================================
 * O16 oracle_replica_search: Alg. 2 Stage 3, expert replication by a search over (expert, rank)
 * candidates (sec. 8.2 prose; listing lines 14-19), ONE instance.
 *   "With Stage 2's placement fixed, P * N_r redundant slots remain.  We allocate them one at a time.
 *    At each step, for every (expert, rank) candidate, we estimate the objective reduction obtained by
 *    adding that replica using a locality-aware token assignment heuristic: tokens prefer same-machine
 *    replicas to avoid cross-machine traffic, and any leftover tokens are routed to minimize per-rank
 *    load.  The candidate yielding the largest reduction is selected.  The loop terminates when all
 *    redundant slots are filled or no candidate improves the objective."
 * Reading 40 fixes what the paper leaves open:
 *   state   every slot j holding expert e carries flows x[j][m] = tokens of e from the sources of
 *           machine m that j serves; RL[r] = sum over the slots of r (Eq.(4)); LT[i][j] = tokens from
 *           machine i served on machine j (Eq.(5) off the diagonal).  Initially every expert has its
 *           base slot only (Stage 2's result): x[j][m] = c[m][e].
 *   objective  F = a * max_r RL[r] + b * max_{i != j} LT[i][j]  (as O12, reading 33).
 *   estimate of candidate (e, r) -- r has a free redundant slot, does not host e, e has tokens and
 *           fewer than max_copies hosts: ONLY e's tokens are re-assigned (everything else stays), over
 *           hosts(e) + r, by the locality-aware heuristic in ONE pass: commodities (e, m) in descending
 *           count (ties ascending m); commodity (e, m) may use the hosts on machine m if there is one,
 *           else all hosts; its tokens go one at a time to the allowed host whose rank is least loaded
 *           (ties: lowest rank).  Delta = F(after) - F(now).
 *   choice  the smallest Delta; ties: lowest expert id, then lowest rank.  "if Delta >= 0 then break".
 *           The replica goes to r's next free redundant slot and the estimate becomes the state.
 *   at most P * N_r rounds.
 * placed_se: every expert exactly once in the base slots (O12's / O8-Stage-2's output); its redundant
 * slots are not read.  out_se: base slots copied, redundant slots filled or -1.
 * stats (may be NULL): [0] replicas placed, [1] F before, [2] F after.
 * Pins (tests/test_oracle_replica_search.py): every round replayed from the output by an independent
 * Python implementation with the CLOSED-FORM water-fill (another algorithmic form than the unit loop
 * below); F strictly decreasing and equal to a numpy recomputation from the final flows; structure;
 * M = 1 / b = 0 special cases; a hand-worked vector (tests/golden/replica_search_vectors.json).
 * ========================================================================================== */
static int64_t swap_objective(int P, int M, int64_t a, int64_t b, const int64_t *RL, const int64_t *LT);   /* O12, below */

typedef struct {
  int E, P, Ns, Nb, M, R;
  int64_t a, b;
  const int32_t *c_me;      /* [M][E] */
  int32_t *se;              /* [S] current placement */
  int64_t *x;               /* [S][M] flows */
  int64_t *RL;              /* [P] */
  int64_t *LT;              /* [M][M] */
} rs_state_t;

static int64_t rs_objective(const rs_state_t *st, const int64_t *RL, const int64_t *LT) {
  return swap_objective(st->P, st->M, st->a, st->b, RL, LT);
}

/* the locality-aware re-assignment of expert e over its current hosts plus (optionally) rank r_new.
 * Writes RL2 / LT2 (the state with e re-assigned) and xnew[rank][m]; returns F(after). */
static int64_t rs_estimate(const rs_state_t *st, int e, int r_new, int64_t *RL2, int64_t *LT2,
                           int64_t *xnew /* [P][M] */, int32_t *is_host /* [P] */) {
  const int P = st->P, M = st->M, Ns = st->Ns, R = st->R, E = st->E;
  memcpy(RL2, st->RL, sizeof(int64_t) * (size_t)P);
  memcpy(LT2, st->LT, sizeof(int64_t) * (size_t)M * M);
  for (int r = 0; r < P; r++) { is_host[r] = 0; for (int m = 0; m < M; m++) xnew[(size_t)r * M + m] = 0; }
  for (int j = 0; j < P * Ns; j++) {            /* take e's tokens out */
    if (st->se[j] != e) continue;
    const int r = j / Ns;
    is_host[r] = 1;
    for (int m = 0; m < M; m++) {
      RL2[r] -= st->x[(size_t)j * M + m];
      LT2[m * M + r / R] -= st->x[(size_t)j * M + m];
    }
  }
  if (r_new >= 0) is_host[r_new] = 1;
  /* commodities (e, m): descending count, ties ascending m */
  int32_t order[128];
  int n = 0;
  for (int m = 0; m < M; m++) if (st->c_me[(size_t)m * E + e] > 0) order[n++] = m;
  for (int u = 1; u < n; u++) {
    const int m = order[u];
    int v = u;
    while (v > 0 && st->c_me[(size_t)order[v - 1] * E + e] < st->c_me[(size_t)m * E + e]) { order[v] = order[v - 1]; v--; }
    order[v] = m;
  }
  for (int u = 0; u < n; u++) {
    const int m = order[u];
    int local = 0;
    for (int r = m * R; r < (m + 1) * R; r++) local |= is_host[r];
    for (int32_t t = 0; t < st->c_me[(size_t)m * E + e]; t++) {      /* one token at a time */
      int best = -1;
      for (int r = 0; r < P; r++) {
        if (!is_host[r] || (local && r / R != m)) continue;
        if (best < 0 || RL2[r] < RL2[best]) best = r;
      }
      RL2[best] += 1;
      LT2[m * M + best / R] += 1;
      xnew[(size_t)best * M + m] += 1;
    }
  }
  return rs_objective(st, RL2, LT2);
}

int oracle_replica_search(int E, int P, int Nb, int Nr, int M, int max_copies, int64_t a, int64_t b,
                          const int32_t *c_me /* [M][E] */, const int32_t *placed_se, int32_t *out_se,
                          int64_t *stats /* [3] or NULL */) {
  const int Ns = Nb + Nr, S = P * Ns;
  if (M <= 0 || M > 128 || P % M != 0 || max_copies < 1 || a < 0 || b < 0) return ORACLE_BAD_ARG;
  int fault = 0;
  rs_state_t st = {E, P, Ns, Nb, M, P / M, a, b, c_me, out_se, NULL, NULL, NULL};
  int64_t *ctot = (int64_t *)calloc((size_t)E, sizeof(int64_t));
  int32_t *seen = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *nhost = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *nred = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int32_t *is_host = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int64_t *RL2 = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  int64_t *LT2 = (int64_t *)calloc((size_t)M * M, sizeof(int64_t));
  int64_t *xnew = (int64_t *)calloc((size_t)P * M, sizeof(int64_t));
  st.x = (int64_t *)calloc((size_t)S * M, sizeof(int64_t));
  st.RL = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  st.LT = (int64_t *)calloc((size_t)M * M, sizeof(int64_t));
  for (int j = 0; j < S; j++) out_se[j] = -1;
  if (!ctot || !seen || !nhost || !nred || !is_host || !RL2 || !LT2 || !xnew || !st.x || !st.RL || !st.LT) {
    fault = ORACLE_NO_MEM; goto done;
  }
  for (int e = 0; e < E; e++)
    for (int m = 0; m < M; m++) {
      if (c_me[(size_t)m * E + e] < 0) fault |= FAULT_ID_RANGE;
      ctot[e] += c_me[(size_t)m * E + e];
    }
  for (int j = 0; j < S; j++) {
    if (j % Ns >= Nb) continue;                          /* the input's redundant slots are not read */
    const int32_t e = placed_se[j];
    if (e < -1 || e >= E) { fault |= FAULT_SLOT_EXPERT; continue; }
    if (e < 0) continue;
    if (seen[e]) fault |= FAULT_SLOT_EXPERT;
    seen[e] = 1;
  }
  for (int e = 0; e < E; e++) if (!seen[e]) fault |= FAULT_SLOT_EXPERT;
  if (fault) goto done;
  for (int j = 0; j < S; j++) {
    if (j % Ns >= Nb || placed_se[j] < 0) continue;
    const int e = placed_se[j], r = j / Ns;
    out_se[j] = e;
    nhost[e] = 1;
    for (int m = 0; m < M; m++) {
      st.x[(size_t)j * M + m] = c_me[(size_t)m * E + e];
      st.RL[r] += c_me[(size_t)m * E + e];
      st.LT[m * M + r / st.R] += c_me[(size_t)m * E + e];
    }
  }
  const int64_t F0 = rs_objective(&st, st.RL, st.LT);
  int64_t F = F0;
  int placed = 0;
  for (int round = 0; round < P * Nr; round++) {
    int64_t best_delta = 0;
    int best_e = -1, best_r = -1;
    for (int e = 0; e < E; e++) {
      if (ctot[e] <= 0 || nhost[e] >= max_copies) continue;
      for (int r = 0; r < P; r++) {
        if (nred[r] >= Nr) continue;
        int hosted = 0;
        for (int j = r * Ns; j < (r + 1) * Ns; j++) hosted |= (out_se[j] == e);
        if (hosted) continue;
        const int64_t delta = rs_estimate(&st, e, r, RL2, LT2, xnew, is_host) - F;
        if (delta < best_delta) { best_delta = delta; best_e = e; best_r = r; }   /* strict: first wins ties */
      }
    }
    if (best_e < 0) break;                                /* "if Delta >= 0 then break" */
    F = rs_estimate(&st, best_e, best_r, RL2, LT2, xnew, is_host);
    out_se[best_r * Ns + Nb + nred[best_r]] = best_e;
    nred[best_r] += 1;
    nhost[best_e] += 1;
    memcpy(st.RL, RL2, sizeof(int64_t) * (size_t)P);
    memcpy(st.LT, LT2, sizeof(int64_t) * (size_t)M * M);
    for (int j = 0; j < S; j++) {
      if (out_se[j] != best_e) continue;
      for (int m = 0; m < M; m++) st.x[(size_t)j * M + m] = xnew[(size_t)(j / Ns) * M + m];
    }
    placed++;
  }
  if (stats) { stats[0] = placed; stats[1] = F0; stats[2] = F; }
done:
  if (fault > 0) for (int j = 0; j < S; j++) out_se[j] = -1;
  free(ctot); free(seen); free(nhost); free(nred); free(is_host); free(RL2); free(LT2); free(xnew);
  free(st.x); free(st.RL); free(st.LT);
  return fault;
}

/* ==========================================================================================
 * O15 oracle_quota_tradeoff: per-source Stage 4 under the objective of Eq.(10),
 *     F = a * L* + b * C*,   L* = max_r L_r (Eq.(4)),  C* = max_{i != j} C_{i,j} (Eq.(5)),
 * with caller-supplied non-negative integers a ~ n1*K1, b ~ n2*K2 (the paper
 * never prints the coefficients: DESIGN.md reading 33).  The paper solves this LP with HiGHS; its
 * only algorithmic description of a locality / load trade-off is the heuristic of PAPER.md:337
 * ("tokens prefer same-machine replicas ..., any leftover tokens are routed to minimize per-rank
 * load").  Reading 39 turns that sentence into a FAMILY of exact sub-problems indexed by a
 * threshold theta and lets the objective choose among them:
 *   member theta: commodity (e, m) whose machine m holds n_loc >= 1 copies of e (ranks) keeps to
 *     those local copies unless serving it locally would by itself put more than theta times the
 *     mean rank load on each of them,
 *         c[e][m] / n_loc  >  theta * total / P      (exact:  c * den * P > num * n_loc * total),
 *     in which case it may use every copy of e ("leftover tokens"); a commodity without a local
 *     copy uses every copy (as in O11).  theta = infinity (den = 0) is O11's hard locality;
 *     theta = 0 lets every non-empty commodity use every copy (the unrestricted min L_max).
 *   Within a member, L_max is minimised exactly by O2 on the virtual instance (as O11).
 *   Result: the member with the smallest F; ties to the earliest member of the ladder.
 * Ladder given by the caller as (num_k, den_k), k = 0 .. n_theta-1.
 * Outputs: member index, F of every member, and q_src / rank_load / traffic / quota_v /
 * slot_off_v / se_v of the chosen member (layouts of O11).
 * Pins (tests/test_oracle_tradeoff.py): member infinity == O11, member 0 reaches O2's optimum on
 * the summed counts; L_max non-increasing along a descending ladder; F_sel = min_k F_k recomputed
 * from the members' outputs with numpy; F_sel >= LP* of Eq.(10) incl. the C rows (HiGHS) and >=
 * the brute-force integer optimum on tiny instances (== when b = 0); a hand-worked vector in
 * which an intermediate theta wins (tests/golden/tradeoff_vectors.json).
 * ========================================================================================== */
int oracle_local_placement_theta(int E, int P, int Ns, int M, int64_t num, int64_t den,
                                 const int32_t *c_v /* [E*M] */, const int32_t *slot_expert,
                                 int32_t *slot_expert_v /* [P*Ns*M] */) {
  const int S = P * Ns;
  if (M <= 0 || P % M != 0 || num < 0 || den < 0) return ORACLE_BAD_ARG;
  const int R = P / M;
  int fault = 0;
  int64_t total = 0;
  for (int v = 0; v < E * M; v++) total += c_v[v];
  for (int j = 0; j < S; j++) {
    const int32_t e = slot_expert[j];
    if (e < -1 || e >= E) fault |= FAULT_SLOT_EXPERT;
    for (int m = 0; m < M; m++) {
      int32_t v = -1;
      if (e >= 0 && e < E) {
        const int mj = (j / Ns) / R;               /* machine of slot j */
        int n_loc = 0;                             /* ranks of machine m that hold e */
        for (int r = m * R; r < (m + 1) * R; r++) {
          int holds = 0;
          for (int j2 = r * Ns; j2 < (r + 1) * Ns; j2++) holds |= (slot_expert[j2] == e);
          n_loc += holds;
        }
        int spill = 0;
        if (n_loc > 0 && den > 0)
          spill = (int64_t)c_v[e * M + m] * den * P > num * n_loc * total;
        if (mj == m || n_loc == 0 || spill) v = e * M + m;
      }
      slot_expert_v[(size_t)j * M + m] = v;
    }
  }
  return fault;
}

int oracle_quota_tradeoff(int E, int P, int Ns, int M, int64_t a, int64_t b, int n_theta,
                          const int64_t *theta_num, const int64_t *theta_den,
                          const int32_t *w_se /* [P][E] per-source counts */, const int32_t *slot_expert,
                          int32_t *member /* [1] */, int64_t *F /* [n_theta] */,
                          int32_t *q_src /* [M][S] */, int32_t *rank_load /* [P] */,
                          int32_t *traffic /* [M][M] */, int32_t *quota_v /* [S*M] */,
                          int32_t *slot_off_v /* [S*M+1] */, int32_t *se_v_sel /* [S*M] */) {
  const int S = P * Ns;
  if (M <= 0 || P % M != 0 || n_theta <= 0 || a < 0 || b < 0) return ORACLE_BAD_ARG;
  const int R = P / M;
  int32_t *c_v = (int32_t *)calloc((size_t)E * M, sizeof(int32_t));
  int32_t *se_v = (int32_t *)calloc((size_t)S * M, sizeof(int32_t));
  int32_t *q_v = (int32_t *)calloc((size_t)S * M, sizeof(int32_t));
  int32_t *so_v = (int32_t *)calloc((size_t)S * M + 1, sizeof(int32_t));
  int32_t *rl = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  int fault = 0, best = -1;
  if (!c_v || !se_v || !q_v || !so_v || !rl) { fault = ORACLE_NO_MEM; goto done; }
  for (int s = 0; s < P; s++)
    for (int e = 0; e < E; e++) c_v[e * M + s / R] += w_se[(size_t)s * E + e];
  for (int k = 0; k < n_theta; k++) {
    int f = oracle_local_placement_theta(E, P, Ns, M, theta_num[k], theta_den[k], c_v, slot_expert, se_v);
    if (f < 0) { fault = f; goto done; }
    f |= oracle_quota(E * M, P, Ns * M, c_v, se_v, q_v, rl, so_v, 3, NULL);
    if (f < 0) { fault = f; goto done; }
    fault |= f;
    int64_t lmax = 0, cmax = 0;
    for (int r = 0; r < P; r++) if (rl[r] > lmax) lmax = rl[r];
    for (int i = 0; i < M; i++)
      for (int mj = 0; mj < M; mj++) {
        if (i == mj) continue;
        int64_t t = 0;
        for (int j = mj * R * Ns; j < (mj + 1) * R * Ns; j++) t += q_v[(size_t)j * M + i];
        if (t > cmax) cmax = t;
      }
    F[k] = a * lmax + b * cmax;
    if (best < 0 || F[k] < F[best]) {              /* strict: ties stay with the earlier member */
      best = k;
      for (int m = 0; m < M; m++)
        for (int j = 0; j < S; j++) q_src[(size_t)m * S + j] = q_v[(size_t)j * M + m];
      for (int i = 0; i < M; i++)
        for (int mj = 0; mj < M; mj++) {
          int64_t t = 0;
          for (int j = mj * R * Ns; j < (mj + 1) * R * Ns; j++) t += q_v[(size_t)j * M + i];
          traffic[i * M + mj] = (int32_t)t;
        }
      memcpy(rank_load, rl, sizeof(int32_t) * (size_t)P);
      memcpy(quota_v, q_v, sizeof(int32_t) * (size_t)S * M);
      memcpy(slot_off_v, so_v, sizeof(int32_t) * ((size_t)S * M + 1));
      memcpy(se_v_sel, se_v, sizeof(int32_t) * (size_t)S * M);
    }
  }
  *member = best;
done:
  free(c_v); free(se_v); free(q_v); free(so_v); free(rl);
  return fault;
}

/* ==========================================================================================
 * NEXT row (second half): Alg. 2 Stage 2, expert relocation by swaps
 * (sec. 8.2 prose; listing lines 4-12).
 *
 * O12 oracle_swap_relocation, ONE (micro-step, layer) instance.  Every expert sits in exactly one
 * base slot (A^{(i)} <- A_base, line 2); rank loads RL[r] = L_r and traffic LT[i][j] = C_{i,j}
 * (Eq.(4)/(5) with one host per expert) are initialised from the placement and the per-source-
 * machine loads c[m][e] (line 3).  Each round (lines 5-12):
 *   h = argmax_r RL[r]                                             "bottleneck rank" (ties: lowest rank)
 *   for each r_l != h: "evaluate swapping a top-K heaviest expert on h with a top-K lightest
 *   expert on r_l": window of `win` experts on each side (heaviest: descending load, ties
 *   ascending id; lightest: ascending load, ties ascending id);
 *   Delta = change of the layer-time objective  F = a * max_r RL[r] + b * max_{i != j} LT[i][j]
 *   (Eq.(3) without its constants: a stands for n1*K1, b for n2*K2, caller-supplied integers --
 *   the paper never prints them, reading 33);
 *   the swap minimising Delta wins (ties: first in the order r_l ascending, then the heaviest-
 *   window order, then the lightest-window order); "if Delta >= 0 then break"; else the two
 *   experts exchange their slots and RL, LT are updated.
 * At most max_rounds rounds ("maximum round count").  Redundant slots are copied
 * unchanged from base_se (Stage 3 fills them later).
 * stats (may be NULL): [0] rounds applied, [1..2] objective before / after (int64 as two int32 is
 * avoided: written as int64_t stats[3]).
 * Pins (tests/test_oracle_swap.py): hand-worked vectors (tests/golden/swap_vectors.json); the
 * objective strictly decreases per applied swap (replayed from the placements with numpy);
 * termination = no improving swap in the bottleneck's window (independent enumeration); structure;
 * balanced input => unchanged; win covering all experts + P = 2 => each round takes the best of
 * all swaps (brute force).
 * ========================================================================================== */
static int64_t swap_objective(int P, int M, int64_t a, int64_t b, const int64_t *RL, const int64_t *LT) {
  int64_t lmax = 0, cmax = 0;
  for (int r = 0; r < P; r++) if (RL[r] > lmax) lmax = RL[r];
  for (int i = 0; i < M; i++)
    for (int j = 0; j < M; j++)
      if (i != j && LT[i * M + j] > cmax) cmax = LT[i * M + j];
  return a * lmax + b * cmax;
}

int oracle_swap_relocation(int E, int P, int Nb, int Nr, int M, int win, int max_rounds, int64_t a,
                           int64_t b, const int32_t *c_me /* [M][E] */, const int32_t *base_se,
                           int32_t *out_se, int64_t *stats /* [3] or NULL */) {
  const int Ns = Nb + Nr, S = P * Ns;
  if (M <= 0 || P % M != 0 || win <= 0 || max_rounds < 0 || a < 0 || b < 0) return ORACLE_BAD_ARG;
  const int R = P / M;
  int fault = 0;
  for (int j = 0; j < S; j++) out_se[j] = base_se[j];
  int64_t *c = (int64_t *)calloc((size_t)E, sizeof(int64_t));
  int32_t *slot_of = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int64_t *RL = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  int64_t *LT = (int64_t *)calloc((size_t)M * M, sizeof(int64_t));
  int64_t *RL2 = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  int64_t *LT2 = (int64_t *)calloc((size_t)M * M, sizeof(int64_t));
  int32_t *heavy = (int32_t *)calloc((size_t)Nb, sizeof(int32_t));
  int32_t *light = (int32_t *)calloc((size_t)Nb, sizeof(int32_t));
  if (!c || !slot_of || !RL || !LT || !RL2 || !LT2 || !heavy || !light) { fault = ORACLE_NO_MEM; goto done; }
  for (int e = 0; e < E; e++) {
    slot_of[e] = -1;
    for (int m = 0; m < M; m++) {
      if (c_me[(size_t)m * E + e] < 0) fault |= FAULT_ID_RANGE;
      c[e] += c_me[(size_t)m * E + e];
    }
  }
  for (int j = 0; j < S; j++) {
    const int32_t e = base_se[j];
    if (e < -1 || e >= E) { fault |= FAULT_SLOT_EXPERT; continue; }
    if (e < 0 || j % Ns >= Nb) continue;                  /* only base slots take part */
    if (slot_of[e] >= 0) fault |= FAULT_SLOT_EXPERT;      /* expert twice in base slots */
    slot_of[e] = j;
  }
  for (int e = 0; e < E; e++) if (slot_of[e] < 0) fault |= FAULT_SLOT_EXPERT;
  if (fault) goto done;
  for (int e = 0; e < E; e++) {                           /* line 3 */
    const int r = slot_of[e] / Ns;
    RL[r] += c[e];
    for (int i = 0; i < M; i++) LT[i * M + r / R] += c_me[(size_t)i * E + e];
  }
  const int64_t F0 = swap_objective(P, M, a, b, RL, LT);
  int64_t F = F0;
  int rounds = 0;
  for (int round = 0; round < max_rounds; round++) {
    int h = 0;
    for (int r = 1; r < P; r++) if (RL[r] > RL[h]) h = r;
    /* window on h: the `win` heaviest experts, descending load, ties ascending id */
    int nh = 0;
    for (int k = 0; k < win && k < Nb; k++) {
      int best = -1;
      for (int j = h * Ns; j < h * Ns + Nb; j++) {
        const int e = out_se[j];
        int taken = 0;
        if (e < 0) continue;
        for (int q = 0; q < nh; q++) taken |= (heavy[q] == e);
        if (taken) continue;
        if (best < 0 || c[e] > c[best] || (c[e] == c[best] && e < best)) best = e;
      }
      if (best < 0) break;
      heavy[nh++] = best;
    }
    int64_t best_delta = 0;
    int best_eh = -1, best_el = -1;
    for (int rl = 0; rl < P; rl++) {
      if (rl == h) continue;
      int nl = 0;                                         /* the `win` lightest experts on r_l */
      for (int k = 0; k < win && k < Nb; k++) {
        int best = -1;
        for (int j = rl * Ns; j < rl * Ns + Nb; j++) {
          const int e = out_se[j];
          int taken = 0;
          if (e < 0) continue;
          for (int q = 0; q < nl; q++) taken |= (light[q] == e);
          if (taken) continue;
          if (best < 0 || c[e] < c[best] || (c[e] == c[best] && e < best)) best = e;
        }
        if (best < 0) break;
        light[nl++] = best;
      }
      for (int x = 0; x < nh; x++)
        for (int y = 0; y < nl; y++) {
          const int eh = heavy[x], el = light[y];
          memcpy(RL2, RL, sizeof(int64_t) * (size_t)P);
          memcpy(LT2, LT, sizeof(int64_t) * (size_t)M * M);
          RL2[h] += c[el] - c[eh];
          RL2[rl] += c[eh] - c[el];
          for (int i = 0; i < M; i++) {
            LT2[i * M + h / R] += (int64_t)c_me[(size_t)i * E + el] - c_me[(size_t)i * E + eh];
            LT2[i * M + rl / R] += (int64_t)c_me[(size_t)i * E + eh] - c_me[(size_t)i * E + el];
          }
          const int64_t delta = swap_objective(P, M, a, b, RL2, LT2) - F;
          if (delta < best_delta) { best_delta = delta; best_eh = eh; best_el = el; }   /* strict: first wins ties */
        }
    }
    if (best_eh < 0) break;                               /* "if Delta >= 0 then break" */
    {
      const int jh = slot_of[best_eh], jl = slot_of[best_el];
      const int rl = jl / Ns;
      RL[h] += c[best_el] - c[best_eh];
      RL[rl] += c[best_eh] - c[best_el];
      for (int i = 0; i < M; i++) {
        LT[i * M + h / R] += (int64_t)c_me[(size_t)i * E + best_el] - c_me[(size_t)i * E + best_eh];
        LT[i * M + rl / R] += (int64_t)c_me[(size_t)i * E + best_eh] - c_me[(size_t)i * E + best_el];
      }
      out_se[jh] = best_el; out_se[jl] = best_eh;
      slot_of[best_eh] = jl; slot_of[best_el] = jh;
      F += best_delta;
      rounds++;
    }
  }
  if (stats) { stats[0] = rounds; stats[1] = F0; stats[2] = F; }
done:
  if (fault > 0) for (int j = 0; j < S; j++) out_se[j] = -1;
  free(c); free(slot_of); free(RL); free(LT); free(RL2); free(LT2); free(heavy); free(light);
  return fault;
}

/* ==========================================================================================
 * O14 oracle_base_placement_machines: Stage 1 in full, Alg. 1 for ONE layer.
 *   lines 1-3   wbar_e = sum_s wbar_{s,e}; experts in descending wbar_e (ties ascending id);
 *               ML[m] = MC[m] = 0;
 *   lines 5-12  machine-level placement: for each expert in that order,
 *                 Delta_{m,e} = sum_{s: machine(s) != m} wbar_{s,e}   (tokens reaching e from other machines)
 *                 score(m,e)  = a * (ML[m] + wbar_e) + b * (MC[m] + Delta_{m,e})   (a ~ n1*K1, b ~ n2*K2)
 *                 m* = argmin score over the machines that still have a free base slot (capacity
 *                 R * N_b; ties lowest m); ML[m*] += wbar_e; MC[m*] += Delta_{m*,e};
 *   lines 13-21 rank-level placement: inside each machine, its experts in descending wbar_e to the
 *               least-loaded local rank with a free base slot (LPT; O7's loop, ties lowest rank).
 * Only the machine of a source matters for Delta, so the input is wbar aggregated per source
 * machine: tot_me[m][e] (readings 21, 33, 37).  With M = 1 this is O7.
 * Pins (tests/test_oracle_placement.py): M = 1 equals O7; the greedy choices replayed step by
 * step in Python from the output; b = 0 => machines balanced as LPT with capacity; a = 0 => every
 * expert on a machine minimising accumulated inbound traffic; hand-worked vector; structure.
 * ========================================================================================== */
int oracle_base_placement_machines(int E, int P, int Nb, int Nr, int M, int64_t a, int64_t b,
                                   const int64_t *tot_me /* [M][E] */, int32_t *slot_expert) {
  const int Ns = Nb + Nr, S = P * Ns;
  int fault = 0;
  for (int j = 0; j < S; j++) slot_expert[j] = -1;
  if (M <= 0 || P % M != 0 || a < 0 || b < 0) return ORACLE_BAD_ARG;
  if ((int64_t)P * Nb < E) return FAULT_SLOT_EXPERT;
  const int R = P / M;
  int64_t *tot = (int64_t *)calloc((size_t)E, sizeof(int64_t));
  int32_t *order = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int32_t *mach = (int32_t *)calloc((size_t)E, sizeof(int32_t));
  int64_t *ML = (int64_t *)calloc((size_t)M, sizeof(int64_t));
  int64_t *MC = (int64_t *)calloc((size_t)M, sizeof(int64_t));
  int32_t *cnt = (int32_t *)calloc((size_t)M, sizeof(int32_t));
  int64_t *RL = (int64_t *)calloc((size_t)P, sizeof(int64_t));
  int32_t *nb = (int32_t *)calloc((size_t)P, sizeof(int32_t));
  if (!tot || !order || !mach || !ML || !MC || !cnt || !RL || !nb) { fault = ORACLE_NO_MEM; goto done; }
  for (int e = 0; e < E; e++) {
    order[e] = e;
    for (int m = 0; m < M; m++) {
      if (tot_me[(size_t)m * E + e] < 0) fault |= FAULT_ID_RANGE;
      tot[e] += tot_me[(size_t)m * E + e];                                        /* line 1 */
    }
  }
  if (fault) goto done;
  for (int x = 1; x < E; x++) {                                                   /* line 2 */
    int32_t e = order[x];
    int y = x;
    while (y > 0 && heavier(tot, e, order[y - 1])) { order[y] = order[y - 1]; y--; }
    order[y] = e;
  }
  for (int x = 0; x < E; x++) {                                                   /* lines 5-12 */
    const int e = order[x];
    int best = -1;
    int64_t best_score = 0;
    for (int m = 0; m < M; m++) {
      if (cnt[m] >= R * Nb) continue;
      const int64_t delta = tot[e] - tot_me[(size_t)m * E + e];
      const int64_t score = a * (ML[m] + tot[e]) + b * (MC[m] + delta);
      if (best < 0 || score < best_score) { best = m; best_score = score; }
    }
    mach[e] = best;
    cnt[best] += 1;
    ML[best] += tot[e];
    MC[best] += tot[e] - tot_me[(size_t)best * E + e];
  }
  for (int x = 0; x < E; x++) {                                                   /* lines 13-21 */
    const int e = order[x], m = mach[e];
    int best = -1;
    for (int r = m * R; r < (m + 1) * R; r++)
      if (nb[r] < Nb && (best < 0 || RL[r] < RL[best])) best = r;
    slot_expert[best * Ns + nb[best]] = e;
    nb[best] += 1;
    RL[best] += tot[e];
  }
done:
  free(tot); free(order); free(mach); free(ML); free(MC); free(cnt); free(RL); free(nb);
  return fault;
}
