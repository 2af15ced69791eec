/*
 * foremoe.h -- C ABI of the B200 (sm_100a) library for the data-parallel hot path behind
 * ForeMoE's micro-step MoE load balancing (arxiv/paper_2606_11867).
 *
 * Given the routing foresight recorded at rollout (top-K expert ids + gate weights per token per
 * MoE layer, PAPER.md:112 sec. 4, :130 sec. 5), micro-step boundaries (sec. 2.3) and a
 * step-level expert placement with replica slots over P logical EP ranks (x_{e,j}, PAPER.md:249
 * sec. 7.2), the library computes on ONE GPU
 *   (1) the per-(micro-step, layer) expert load histogram  w_{s,e}  (PAPER.md:204 Table 1, :247),
 *   (2) Stage 4 "token assignment" with the placement fixed (sec. 8.2 Eq.(10);
 *       water-filling variant PAPER.md:821-828 Alg. 3 lines 18-21, :844-846 App. D) as integer
 *       per-slot quotas, and the slot of every (token, k) pair,
 *   (3) the dispatch realising the plan (PAPER.md:58 sec. 2.1, :427 sec. 9): stable counting-sort
 *       permutation + offsets, row gather into contiguous per-rank / per-slot buffers, and the
 *       inverse weighted top-K combine (sec. 2.1).
 *
 * Notation (Table 1): L MoE layers, E experts, K top-k, P logical ranks,
 * Ns = Nb + Nr slots per rank (Nb = E / P base, Nr redundant), S = P * Ns global slots, slot j
 * belongs to rank j / Ns, T tokens in the step, micro-step i = tokens [mb_off[i], mb_off[i+1]),
 * T_i its token count, H hidden size.  instance = one (micro-step, layer).  pair = one
 * (token, k) entry; pair p = t * K + k is the LAYER-GLOBAL pair index.  The dispatched rows of
 * layer l form one array of T * K rows; instance (i, l) owns rows [mb_off[i]*K, mb_off[i+1]*K),
 * ordered by rank, then by slot, stable in (t, k) order inside a slot (reading 13).
 *
 * General rules
 *  - Every data pointer is a DEVICE pointer owned by the caller unless the argument is marked
 *    "host".  The foremoe_shape_t pointer is a host pointer, read during the call only.
 *  - The library allocates no device memory, keeps no tunable global state and is re-entrant: any
 *    number of host threads may drive any number of streams and devices concurrently.  Its only
 *    process state is a lock-free memo of launch facts (SM count, occupancy, shared-memory opt-in)
 *    per device and kernel variant, filled on first use or by foremoe_warmup.
 *    All entry points except foremoe_workspace_bytes / foremoe_version / foremoe_warmup /
 *    foremoe_step_host enqueue work on `stream` (a cudaStream_t passed as void*) and return without
 *    synchronising.
 *  - Return value: FOREMOE_OK, or a negative host-detectable error (nothing was enqueued).
 *  - Stream order is the only ordering the data-path calls need: their kernels are launched with
 *    programmatic stream serialisation and, by default, read nothing from global memory before the
 *    grid dependency is resolved, so inputs written by the preceding kernel of the stream (inv by
 *    foremoe_assign, x / expert_out / w by the caller's kernels) are always seen complete.
 *    shape.flags = FOREMOE_FLAG_PLAN_STABLE is the caller's promise that the PLAN arrays of the call
 *    (mb_off, inv, w) are not written by the kernel launched immediately before it on the same
 *    stream -- foremoe_assign excepted: it ends with a full serialisation point, so calling the data
 *    path right after it is covered.  The data-path kernels then fetch their first plan entries
 *    while the preceding kernel drains (activations are still only touched after the dependency);
 *    worth 4 % at one-sample micro-steps, under 1 % at 16 K tokens (profiles/r02_sweeps.md).
 *    The promise covers ONE kernel back because the library's own kernels release their dependents
 *    only after their own grid-dependency wait has returned: in  [kernel that writes w] ->
 *    foremoe_dispatch -> foremoe_combine(PLAN_STABLE)  the combine cannot start before the writer
 *    has completed, although the dispatch between them never touches w (tests/test_gpu_pdl_chain.py).
 *    If the kernel launched immediately before the call is the CALLER's and itself uses programmatic
 *    dependent launch, it must do the same (griddepcontrol.wait before .launch_dependents), or the
 *    promise has to extend to whatever that kernel was allowed to overlap.
 *  - CUDA graphs: the data-path calls (dispatch, combine, *_bwd) are stream-capturable.  The first
 *    launch of a kernel variant on a device queries occupancy and opts into large shared memory,
 *    which capture does not allow: call foremoe_warmup(shape) once per shape and device before
 *    capturing (or run the calls once eagerly).
 *  - Data-dependent faults cannot be seen without a sync; they are OR-ed into *dev_status
 *    (device int32, may be NULL, never cleared by the library): FOREMOE_FAULT_* bits.  On a
 *    device fault the affected instance's outputs are unspecified, all writes stay in bounds.
 *  - Requirements: 0 <= T, T * K < 2^31 (T = 0, a step without tokens, is valid: the [L][T][K] arrays
 *    are then empty and may be NULL); 1 <= K <= 32, K <= E; E % P == 0 and Nb == E / P; Nr >= 0;
 *    row bytes H * es (es = 2 for bf16, 4 for fp32) a multiple of 16; x / buf / expert_out / y
 *    16-byte aligned; int32 / fp32 arrays 4-byte aligned (K = 10 id rows are only 8-byte
 *    aligned -- nothing wider is assumed).
 */
#ifndef FOREMOE_H_
#define FOREMOE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FOREMOE_OK 0
#define FOREMOE_ERR_INVALID_ARG (-1)      /* NULL, bad dims, misaligned pointer, bad mb range */
#define FOREMOE_ERR_WORKSPACE (-2)        /* workspace_bytes too small                        */
#define FOREMOE_ERR_CUDA (-3)             /* CUDA error at launch / copy                      */

#define FOREMOE_FAULT_ID_RANGE 1          /* expert id outside [0, E) (pair ignored)          */
#define FOREMOE_FAULT_NO_HOST 2           /* expert with tokens but no slot: Eq.(7) violated,
                                             or hist inconsistent with ids                    */
#define FOREMOE_FAULT_SLOT_EXPERT 4       /* slot_expert value outside [-1, E)                */
#define FOREMOE_FAULT_MB_OFF 8            /* mb_off not non-decreasing or not 0 .. T          */
#define FOREMOE_FAULT_QUOTA_IN 16         /* caller quota violates Eq.(8)/(9) or is negative  */
#define FOREMOE_FAULT_SOURCE 32           /* tok_src value outside [0, P)                     */

#define FOREMOE_ACT_BF16 0
#define FOREMOE_ACT_FP32 1

#define FOREMOE_FLAG_PLAN_STABLE 1  /* see "Stream order" above                                    */

typedef struct {
  int32_t L, E, K;             /* MoE layers, experts, top-k                                   */
  int32_t P, Nb, Nr;           /* logical ranks, base / redundant slots per rank               */
  int32_t T, n_mb;             /* tokens in the step, micro-steps                              */
  int32_t H, act_dtype;        /* hidden size; FOREMOE_ACT_BF16 / FOREMOE_ACT_FP32             */
  int32_t placement_mb_stride; /* 0: slot_expert is [L][S] (step-level placement);
                                  L*S: slot_expert is [n_mb][L][S] (one placement per micro-step,
                                  PAPER.md:343 A^{(i)})                                         */
  int32_t flags;               /* 0, or FOREMOE_FLAG_PLAN_STABLE                               */
} foremoe_shape_t;

/* Library version (major * 100 + minor).  Host only. */
int foremoe_version(void);

/* Bytes of device scratch foremoe_assign needs for this shape.  Host only, no CUDA call. */
int foremoe_workspace_bytes(const foremoe_shape_t *shape, size_t *bytes /* host, out */);

/*
 * Prepares every data-path kernel variant this shape selects (dispatch, combine, combine_bwd with and
 * without dw, dispatch_bwd) on the calling thread's current device: opts them into large shared
 * memory and memoises their occupancy.  Launches nothing and does not synchronise; `stream` is
 * accepted for symmetry and ignored.  After it, the data-path calls for this shape issue no CUDA
 * call other than the kernel launch, so the very first one may already be stream-captured.
 * Optional otherwise: every call prepares its own variant on first use.
 */
int foremoe_warmup(const foremoe_shape_t *shape, void *stream);

/*
 * (a1) Load histogram -- w_{s,e} with the single source rank and its step
 * aggregate (sec. 8.1).
 *   ids       [L][T][K] int32, expert ids of the routing trace (layer-major).
 *   mb_off    [n_mb+1]  int32, micro-step token boundaries, mb_off[0] = 0, mb_off[n_mb] = T.
 *   hist      [n_mb][L][E] int32 out: hist[i][l][e] = #{(t,k): t in micro-step i, ids[l][t][k] == e}.
 *   step_hist [L][E] int64 out, or NULL: sum over micro-steps.
 * Faults: ID_RANGE (the pair is not counted), MB_OFF (hist and step_hist are all zero).
 */
int foremoe_load_hist(const foremoe_shape_t *shape, const int32_t *ids, const int32_t *mb_off,
                      int32_t *hist, int64_t *step_hist, int32_t *dev_status, void *stream);

/*
 * (a2-a4) Stage-4 token assignment for every instance of the step, placement fixed.
 *   hist        [n_mb][L][E] from foremoe_load_hist on the same ids / mb_off.
 *   slot_expert [L][S] (or [n_mb][L][S], see placement_mb_stride) int32: expert held by global
 *               slot j = rank * Ns + local; -1 = empty slot (reading 9).
 *   quota_in    NULL: quotas are computed by the exact water-filling rule (O2):
 *               forced loads, Gauss-Seidel water-filling passes to a fixpoint (PAPER.md:826-827,
 *               :844-846), unit augmentations until max rank load is optimal.
 *               else [n_mb][L][S] caller-supplied quotas (e.g. from an LP of Eq.(10)), validated
 *               against Eq.(8) conservation and Eq.(9) feasibility.
 *   quota       [n_mb][L][S]   out: tokens each slot receives.
 *   rank_load   [n_mb][L][P]   out: L_r of Eq.(4) = sum of the quotas of rank r's slots.
 *   slot_off    [n_mb][L][S+1] out: exclusive prefix of quota (rows of slot j inside the instance).
 *   pair_slot   [L][T][K]      out: global slot of every pair: the pair with stable rank n among
 *               the instance's pairs of expert e goes to the host slot of e (ascending slot index)
 *               whose cumulative-quota interval contains n (reading 1).  -1 on fault.
 *   inv         [L][T][K]      out: layer-global destination row of every pair
 *               = mb_off[i]*K + slot_off[j] + (stable rank of the pair inside slot j).  -1 on fault.
 *   workspace   device scratch of at least foremoe_workspace_bytes() bytes, 16-byte aligned.
 * pair_slot and inv may BOTH be NULL: only the quotas (a2) are computed -- quota, rank_load,
 * slot_off -- and the ids are not read (used to evaluate candidate placements, see
 * foremoe_tradeoff_select).
 * Faults: ID_RANGE, NO_HOST, SLOT_EXPERT, MB_OFF, QUOTA_IN.
 */
int foremoe_assign(const foremoe_shape_t *shape, const int32_t *ids, const int32_t *mb_off,
                   const int32_t *hist, const int32_t *slot_expert, const int32_t *quota_in,
                   int32_t *quota, int32_t *rank_load, int32_t *slot_off, int32_t *pair_slot,
                   int32_t *inv, void *workspace, size_t workspace_bytes, int32_t *dev_status,
                   void *stream);

/*
 * (a1-a4) foremoe_load_hist followed by foremoe_assign as ONE call that passes over the ids twice
 * instead of three times: the first pass counts every ranking chunk (a run of consecutive tokens of
 * one instance), the instance histogram w_{s,e} is the sum of its chunks'
 * counts and is written to `hist` before the quotas are computed from it, the second pass ranks the
 * pairs.  Every output is bit-identical to the two separate calls; arguments as there, except that
 * hist [n_mb][L][E] (and step_hist [L][E] or NULL) are OUTPUTS and pair_slot / inv are required.
 * Use it when the placement does not depend on this step's histogram (a given step-level
 * placement); planners that derive the placement from hist / step_hist call the two entry points.
 * Faults: as foremoe_load_hist and foremoe_assign together.
 */
int foremoe_plan(const foremoe_shape_t *shape, const int32_t *ids, const int32_t *mb_off,
                 const int32_t *slot_expert, const int32_t *quota_in, int32_t *hist,
                 int64_t *step_hist, int32_t *quota, int32_t *rank_load, int32_t *slot_off,
                 int32_t *pair_slot, int32_t *inv, void *workspace, size_t workspace_bytes,
                 int32_t *dev_status, void *stream);

/*
 * foremoe_plan for callers that cannot bring a workspace.  Same arguments, outputs, faults and
 * stream behaviour as foremoe_plan, bit for bit, minus `workspace` / `workspace_bytes`.
 *
 * Who needs it: code that runs as a guest inside an engine whose own allocator took (almost) all of
 * the GPU's memory when it started, so that a cudaMalloc of even a few MB fails; a plugin whose host
 * allows device allocation only during initialisation; a step loop that cannot afford the
 * device-wide synchronisation that comes with cudaMalloc / cudaFree.  Such callers already own their
 * inputs and outputs but have nowhere to take the plan kernels' scratch from.
 *
 * Where the scratch lives instead: in ONE array of FOREMOE_NOALLOC_SCRATCH_BYTES (8 MiB) of device
 * global memory that is part of the library image.  Every GPU on which the process uses CUDA while
 * the library is loaded carries those 8 MiB until the process exits, whether or not this call is
 * ever made.  The call itself allocates and frees nothing and calls no library routine that does.
 *
 * Limit: the shape must satisfy foremoe_workspace_bytes(shape) <= FOREMOE_NOALLOC_SCRATCH_BYTES;
 * otherwise the call returns FOREMOE_ERR_WORKSPACE and enqueues nothing (checked on the host before
 * any CUDA call; compare the two numbers yourself to know in advance).  Roughly: n_mb * L * S * 8 +
 * L * (T * K / 4096 + n_mb) * E * 4 bytes -- e.g. E = 128, K = 8, P = 8, Ns = 18, L = 4, 8 micro-steps
 * of 16 K tokens need 0.56 MiB; the 48-layer, 512 K-token config 2 needs 26.5 MiB and must use foremoe_plan.
 *
 * First call on a device: the library looks up the array's address on the calling thread's current
 * device (one cudaGetSymbolAddress, remembered per device; FOREMOE_ERR_CUDA if it fails).  That
 * look-up is a runtime query, not a launch: make the first call on every device an ordinary eager
 * one, before any stream capture begins on that device.  Later calls only launch kernels.
 *
 * Sharing: all calls on one device use the same array, on whatever stream, from whatever thread.
 * Two calls whose kernels can be in flight on the GPU at the same time (different streams without an
 * event between them, or two host threads on two streams) overwrite each other's scratch and both
 * results are garbage without any fault bit: order them yourself.  Calls in one stream are safe
 * back to back.  The array still holds the previous call's tables when the next call starts; that
 * is harmless, because every table is rebuilt before it is read and nothing in it has to start at
 * zero, so the library clears nothing.  Unlike every other entry point, this one is therefore NOT
 * re-entrant across streams.
 */
#define FOREMOE_NOALLOC_SCRATCH_BYTES (8u << 20)
int foremoe_plan_noalloc(const foremoe_shape_t *shape, const int32_t *ids, const int32_t *mb_off,
                         const int32_t *slot_expert, const int32_t *quota_in, int32_t *hist,
                         int64_t *step_hist, int32_t *quota, int32_t *rank_load, int32_t *slot_off,
                         int32_t *pair_slot, int32_t *inv, int32_t *dev_status, void *stream);

/*
 * (a4-a5) Dispatch of micro-steps [mb_begin, mb_end) of one layer: the permutation and the row
 * gather into contiguous per-rank / per-slot buffers.
 *   inv   [L][T][K] from foremoe_assign (the whole array; the call indexes layer / range itself).
 *   x     [T_range][H] activations, row 0 = token mb_off[mb_begin]; bf16 or fp32 per act_dtype.
 *   perm  [T_range*K] int32 out, or NULL: perm[d - row0] = p for the pair p with inv[l][p] = d,
 *         row0 = mb_off[mb_begin]*K (layer-global pair index; stable counting sort by slot).
 *   buf   [T_range*K][H] out: buf[d - row0][:] = x[p / K - mb_off[mb_begin]][:], bitwise copy.
 * Pairs with inv < 0 (faulted in assign) are skipped; their rows of buf are left untouched.
 */
int foremoe_dispatch(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin, int32_t mb_end,
                     const int32_t *mb_off, const int32_t *inv, const void *x, int32_t *perm,
                     void *buf, int32_t *dev_status, void *stream);

/*
 * (a6) Combine of micro-steps [mb_begin, mb_end) of one layer: the weighted top-K sum
 * in fp32 with fused multiply-add, k ascending, from acc = 0 (reading 16):
 *   y[t - t0][h] = fma(w[l][t][K-1], eo[inv[l][t][K-1] - row0][h], ... fma(w[l][t][0], eo[...][h], 0))
 *   w          [L][T][K] fp32 gate weights of the trace (the whole array).
 *   expert_out [T_range*K][H] rows in the order of buf (bf16 or fp32 per act_dtype).
 *   y          [T_range][H] fp32 out.
 * Pairs with inv < 0 contribute nothing.
 */
int foremoe_combine(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin, int32_t mb_end,
                    const int32_t *mb_off, const int32_t *inv, const float *w,
                    const void *expert_out, float *y, int32_t *dev_status, void *stream);

/*
 * (NEXT) Stage 1 base placement at rank level for every layer: experts in
 * descending step load (ties ascending id), each to the least-loaded rank that still has a free
 * base slot (ties lowest rank) -- Alg. 1 lines 13-21 with the N_b capacity of
 * PAPER.md:284; one machine (the machine-level greedy needs coefficients the paper never gives).
 *   step_hist   [L][E] int64 from foremoe_load_hist.
 *   slot_expert [L][S] int32 out: base slots filled front to back, redundant slots -1.
 * Faults: ID_RANGE (negative load or load >= 2^31): that layer's output is all -1.
 */
int foremoe_base_placement(const foremoe_shape_t *shape, const int64_t *step_hist,
                           int32_t *slot_expert, int32_t *dev_status, void *stream);

/*
 * (NEXT) Stage 1 in full -- Alg. 1 with M machines of
 * R = P / M ranks: experts in descending step load; machine-level greedy (lines 5-12)
 *     score(m, e) = a * (ML[m] + w_e) + b * (MC[m] + Delta_{m,e}),  Delta_{m,e} = w_e - w_{m,e}
 * over the machines that still have a free base slot (capacity R * N_b; ties lowest m), with the
 * caller-supplied integers a ~ n1*K1, b ~ n2*K2 in [0, 2^20] (readings 33, 37); then the
 * rank-level LPT of foremoe_base_placement inside every machine (lines 13-21).
 *   step_hist_v [L][E*M] int64: step load of expert e from the sources of machine m at e*M + m
 *               (foremoe_load_hist's step_hist on foremoe_source_ids' output; M = 1: step_hist).
 *   slot_expert [L][S] out.  M <= 64.  Faults: ID_RANGE (negative load): that layer is all -1.
 */
int foremoe_base_placement_machines(const foremoe_shape_t *shape, int32_t M, int64_t a, int64_t b,
                                    const int64_t *step_hist_v, int32_t *slot_expert,
                                    int32_t *dev_status, void *stream);

/*
 * (NEXT) Per-micro-step placement A^{(i)}: Alg. 3 Stages 2-3
 * for every (micro-step, layer) instance.  Machines are M groups of
 * R = P / M consecutive ranks; an expert is local to the machine of its base rank.
 *   Stage 2: local experts in descending micro-step load, each to the least-loaded local rank with
 *            a free base slot.
 *   Stage 3: R * N_r rounds per machine: the locally heaviest expert (largest load per copy, exact;
 *            ties lower id; zero-load experts never) gets a replica on the least-loaded local rank
 *            with a free redundant slot that does not host it yet; rank loads carry the exact
 *            integer even split over an expert's hosts (readings 21-25).
 *   hist             [n_mb][L][E] from foremoe_load_hist.
 *   base_slot_expert [L][S] (e.g. from foremoe_base_placement): defines each expert's machine.
 *   slot_expert_mb   [n_mb][L][S] out: feed it to foremoe_assign with
 *                    shape.placement_mb_stride = L * S.
 * Faults: SLOT_EXPERT (base placement has a bad value, misses an expert, or overfills a machine),
 * ID_RANGE (negative load): that instance's output is all -1.
 */
int foremoe_microstep_placement(const foremoe_shape_t *shape, int32_t M, const int32_t *hist,
                                const int32_t *base_slot_expert, int32_t *slot_expert_mb,
                                int32_t *dev_status, void *stream);

/*
 * (NEXT) Backward of the data path -- the policy-update stage: "the backward
 * pass triggers an additional gradient computation and additional MoE dispatch and MoE combine of
 * gradients" (sec. 7.1, n1 = 3, n2 = 4), on the SAME plan (inv, w) as the forward of
 * the micro-step (PAPER.md:170 Fig. 7, :188).  Same range / row conventions as foremoe_combine.
 *
 * foremoe_combine_bwd -- backward of (a6), the "MoE dispatch of gradients" (token -> slot order):
 *   dy            [T_range][H] fp32: gradient of the loss w.r.t. y.
 *   expert_out    [T_range*K][H] the forward expert outputs (act dtype), or NULL if dw is NULL.
 *   d_expert_out  [T_range*K][H] out (act dtype):
 *                 d_expert_out[inv[l][t][k] - row0][h] = round_act(w[l][t][k] * dy[t - t0][h]):
 *                 one fp32 multiply, then round-to-nearest-even to bf16 when act_dtype is bf16
 *                 (reading 27; NaN payloads unspecified).  Rows no pair maps to
 *                 (faulted pairs) are left untouched.
 *   dw            [L][T][K] fp32 out (the whole array; the call writes layer / range), or NULL:
 *                 dw[l][t][k] = sum_h dy[t - t0][h] * float(expert_out[inv[l][t][k] - row0][h]),
 *                 reduced in fp32 (per-lane fma chains, then a fixed shuffle tree: deterministic,
 *                 within H * 2^-24 * sum_h |dy * eo| of the exact sum); 0 for pairs with inv < 0.
 *
 * foremoe_dispatch_bwd -- backward of (a5), the "MoE combine of gradients" (slot -> token order):
 *   d_buf [T_range*K][H] gradient w.r.t. the dispatched rows (act dtype);
 *   dx    [T_range][H] fp32 out: dx[t - t0][h] = sum_k float(d_buf[inv[l][t][k] - row0][h]),
 *         fp32 adds, k ascending from 0 (= foremoe_combine with unit weights, bit for bit).
 */
int foremoe_combine_bwd(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin, int32_t mb_end,
                        const int32_t *mb_off, const int32_t *inv, const float *w, const float *dy,
                        const void *expert_out, void *d_expert_out, float *dw, int32_t *dev_status,
                        void *stream);

int foremoe_dispatch_bwd(const foremoe_shape_t *shape, int32_t layer, int32_t mb_begin, int32_t mb_end,
                         const int32_t *mb_off, const int32_t *inv, const void *d_buf, float *dx,
                         int32_t *dev_status, void *stream);

/*
 * (NEXT) Per-source, multi-machine Stage 4.  Every token has a source rank
 * (w_{s,e} is a P x E matrix); the P ranks form M machines of R = P / M
 * consecutive ranks; C_{i,j} of Eq.(5) counts the tokens flowing from the ranks of
 * machine i to the slots of machine j.  Token assignment follows the paper's locality-aware
 * heuristic ("tokens prefer same-machine replicas to avoid cross-machine traffic,
 * and any leftover tokens are routed to minimize per-rank load"), made exact like Stage 4 itself
 * (readings 29-31): commodity (e, m) = tokens of expert e from sources on machine m; its
 * allowed hosts are the slots holding e on machine m if there is one, else all slots holding e;
 * among the assignments respecting the allowed hosts, L_max is minimised by the water-filling of
 * foremoe_assign.  The three calls below build the VIRTUAL instance on which the four calls of the
 * hot path then run unchanged:
 *     virtual expert  v = e * M + m                 (E_v = E * M)
 *     virtual slot    j * M + m  on the rank of j   (N_b,v = N_b * M, N_r,v = N_r * M, S_v = S * M)
 *     shape_v = shape with E, Nb, Nr multiplied by M (placement_mb_stride too, if non-zero)
 *   foremoe_source_ids      -> ids_v;   foremoe_local_placement -> slot_expert_v;
 *   foremoe_load_hist(shape_v, ids_v)  -> hist_v[n_mb][L][E*M]: hist_v[..][e*M+m] = w_{m,e} summed over
 *                                         the sources of machine m (with M = P: w_{s,e} itself);
 *   foremoe_assign(shape_v, ids_v, hist_v, slot_expert_v) -> quota_v[n_mb][L][S*M] with
 *       quota_v[..][j*M+m] = tokens of source machine m sent to slot j, rank_load (unchanged
 *       meaning), pair_slot_v = (real slot) * M + (source machine), inv: rows grouped by rank, then
 *       slot, then source machine, stable in (t, k) order;
 *   foremoe_dispatch / foremoe_combine / *_bwd (shape_v): unchanged (they read K, H, T, inv only);
 *   foremoe_traffic(quota_v) -> the M x M traffic matrix of every instance.
 *
 * foremoe_source_ids:  tok_src [T] int32 source rank of every token (the same for all layers);
 *   ids_v [L][T][K] out = ids * M + tok_src[t] / R, or -1 for an id outside [0, E) (fault ID_RANGE)
 *   or a source outside [0, P) (fault SOURCE).  ids_v may not alias ids.
 * foremoe_local_placement: slot_expert [L][S] (or [n_mb][L][S] per placement_mb_stride) ->
 *   slot_expert_v [.][S*M]: v on virtual slot j*M+m iff slot j holds e and (machine(j) == m or
 *   machine m holds no copy of e), else -1.  Fault SLOT_EXPERT for values outside [-1, E).
 * foremoe_traffic: traffic [n_mb][L][M][M] int32 out: traffic[..][i][j] = sum over the slots of
 *   machine j of quota_v[..][slot*M + i]; off-diagonal = C_{i,j} of Eq.(5), diagonal = tokens that
 *   stay inside machine i.  M <= 128.
 * `shape` in all three calls is the REAL shape; M must divide P.
 */
int foremoe_source_ids(const foremoe_shape_t *shape, int32_t M, const int32_t *ids,
                       const int32_t *tok_src, int32_t *ids_v, int32_t *dev_status, void *stream);

int foremoe_local_placement(const foremoe_shape_t *shape, int32_t M, const int32_t *slot_expert,
                            int32_t *slot_expert_v, int32_t *dev_status, void *stream);

int foremoe_traffic(const foremoe_shape_t *shape, int32_t M, const int32_t *quota_v,
                    int32_t *traffic, void *stream);

/*
 * (NEXT, the C* term) Per-source Stage 4 under the objective of Eq.(10),
 *     F = a * L* + b * C*,  L* = max_r L_r,  C* = max_{i != j} C_{i,j},
 * with caller-supplied integers a ~ n1*K1, b ~ n2*K2 in [0, 2^20] (reading 33).  The paper
 * solves this LP on the CPU; here the locality heuristic of PAPER.md:337 becomes a LADDER of exact
 * sub-problems (reading 39): member theta = num / den restricts commodity (e, m) to the
 * copies of e on machine m unless its count per local copy exceeds theta times the mean rank load,
 *     hist_v[e*M+m] * den * P  >  num * n_loc(e, m) * sum(hist_v),
 * in which case (or when machine m holds no copy) it may use every copy.  den = 0 means theta =
 * infinity: foremoe_local_placement's hard locality; num = 0, den = 1: no restriction.
 * Composition (paper_2606_11867_b200/runner.py TradeoffStepPlan), per member k of the ladder:
 *   foremoe_local_placement_theta -> slot_expert_v_k [n_mb][L][S*M]  (one placement per instance)
 *   foremoe_assign(shape_v with placement_mb_stride = L*S*M, pair_slot = inv = NULL) -> quota_k,
 *       rank_load_k  (exact min L_max within the member);  foremoe_traffic -> traffic_k;
 * then foremoe_tradeoff_select picks, per instance, the member with the smallest F (ties: the
 * earliest) and copies out its quotas and placement, and one more foremoe_assign with
 * quota_in = quota_sel on slot_expert_v_sel assigns the pairs.
 *
 * foremoe_local_placement_theta: hist_v [n_mb][L][E*M] (foremoe_load_hist on the commodity ids);
 *   slot_expert [L][S] or [n_mb][L][S] per placement_mb_stride; slot_expert_v_mb [n_mb][L][S*M] out.
 *   theta_num, theta_den in [0, 2^20].  Fault SLOT_EXPERT for values outside [-1, E).
 * foremoe_tradeoff_select: arrays with a leading member axis [n_members][n_mb][L][...]:
 *   rank_load_k [..][P], traffic_k [..][M][M], quota_k [..][S*M], slot_expert_v_k [..][S*M];
 *   member [n_mb][L] out; F [n_members][n_mb][L] int64 out or NULL; quota_sel, slot_expert_v_sel
 *   [n_mb][L][S*M] out.  n_members <= 64, M <= 128.
 * `shape` in both calls is the REAL shape; M must divide P.
 */
int foremoe_local_placement_theta(const foremoe_shape_t *shape, int32_t M, int64_t theta_num,
                                  int64_t theta_den, const int32_t *hist_v, const int32_t *slot_expert,
                                  int32_t *slot_expert_v_mb, int32_t *dev_status, void *stream);

int foremoe_tradeoff_select(const foremoe_shape_t *shape, int32_t M, int32_t n_members, int64_t a,
                            int64_t b, const int32_t *rank_load_k, const int32_t *traffic_k,
                            const int32_t *quota_k, const int32_t *slot_expert_v_k, int32_t *member,
                            int64_t *F, int32_t *quota_sel, int32_t *slot_expert_v_sel, void *stream);

/*
 * (NEXT, second half) Alg. 2 Stage 2: expert relocation by swaps
 * (sec. 8.2; listing lines 4-12) for every (micro-step, layer)
 * instance, starting from the base placement (every expert in exactly one base slot).  Each round:
 * h = the most loaded rank (ties: lowest rank); for every other rank r_l the `win` heaviest experts
 * on h (descending load, ties ascending id) x the `win` lightest experts on r_l (ascending load,
 * ties ascending id); the swap with the smallest change Delta of the layer-time objective
 *     F = a * max_r RL[r] + b * max_{i != j} LT[i][j]          (Eq.(3) without its constants;
 *     a ~ n1*K1, b ~ n2*K2 are caller-supplied integers in [0, 2^20]: DESIGN.md reading 33)
 * wins (ties: first in the order r_l ascending, heaviest-window order, lightest-window order);
 * stop when Delta >= 0 or after max_rounds rounds; otherwise the two experts exchange slots.
 *   hist_v           [n_mb][L][E*M]: load of expert e from the sources of machine m at e*M + m
 *                    (foremoe_load_hist on foremoe_source_ids' output; with M = 1 the plain hist).
 *   base_slot_expert [L][S]; redundant slots are copied through unchanged.
 *   slot_expert_mb   [n_mb][L][S] out (feed it to foremoe_assign with placement_mb_stride = L*S).
 *   rounds           [n_mb][L] out or NULL: swaps applied per instance.
 * Faults: SLOT_EXPERT (base placement has a bad value, or an expert twice / missing in the base
 * slots), ID_RANGE (negative load): that instance's output is all -1.
 */
int foremoe_swap_relocation(const foremoe_shape_t *shape, int32_t M, int32_t win, int32_t max_rounds,
                            int64_t a, int64_t b, const int32_t *hist_v,
                            const int32_t *base_slot_expert, int32_t *slot_expert_mb, int32_t *rounds,
                            int32_t *dev_status, void *stream);

/*
 * (NEXT) Stage 3 alone: replication on per-micro-step placements whose base
 * slots are already final -- the output of foremoe_swap_relocation -- with Alg. 3's choice rule
 * (readings 22-25), so that Alg. 2's relocation by swaps, replication
 * and Stage 4 compose.  (Alg. 2's own replica score, the "estimated drop" under a locality-aware
 * assignment of PAPER.md:337, is foremoe_replica_search below.)
 *   hist                  [n_mb][L][E] micro-step loads.
 *   placed_slot_expert_mb [n_mb][L][S]: every expert exactly once in the base slots; the
 *                         redundant slots of the input are not read.
 *   slot_expert_mb        [n_mb][L][S] out (may alias the input): base slots copied, redundant
 *                         slots filled by R * N_r rounds per machine, -1 where nothing is left.
 * Faults: SLOT_EXPERT, ID_RANGE as in foremoe_microstep_placement (instance output all -1).
 */
int foremoe_replication(const foremoe_shape_t *shape, int32_t M, const int32_t *hist,
                        const int32_t *placed_slot_expert_mb, int32_t *slot_expert_mb,
                        int32_t *dev_status, void *stream);

/*
 * (NEXT) Alg. 2 Stage 3: expert replication by a search over (expert, rank) candidates (PAPER.md:337
 * sec. 8.2; listing lines 14-19) for every (micro-step, layer) instance, on
 * placements whose base slots are final (foremoe_swap_relocation's output).  State: every slot
 * holding expert e carries the tokens of e it serves per source machine; RL[r] (Eq.(4)) and LT[i][j]
 * (Eq.(5)) follow.  Each round, for every candidate (e, r) -- rank r has a free redundant slot, does
 * not host e, e has tokens and fewer than max_copies hosts -- ONLY e's tokens are re-assigned over
 * hosts(e) + r by the locality-aware heuristic ("tokens prefer same-machine replicas ..., any leftover
 * tokens are routed to minimize per-rank load"): commodities (e, m) in descending count (ties
 * ascending m), each over the hosts on machine m if there is one, else all hosts, token by token to
 * the least-loaded allowed rank (ties: lowest rank).  Delta = change of F = a * max_r RL +
 * b * max_{i != j} LT (a, b as in foremoe_swap_relocation).  The smallest Delta wins (ties: lowest
 * expert id, then lowest rank); "if Delta >= 0 then break"; otherwise the replica takes r's next
 * free redundant slot and the estimate becomes the state; at most P * N_r replicas (DESIGN.md
 * reading 40).
 *   hist_v                [n_mb][L][E*M] (as foremoe_swap_relocation).
 *   placed_slot_expert_mb [n_mb][L][S]: every expert exactly once in the base slots; redundant slots
 *                         are not read.
 *   slot_expert_mb        [n_mb][L][S] out (may alias the input): base slots copied, redundant slots
 *                         filled front to back or -1.
 *   replicas              [n_mb][L] out or NULL: replicas placed.
 *   F                     [n_mb][L][2] int64 out or NULL: objective before / after.
 *   M <= 32, 1 <= max_copies <= 31.
 * Faults: SLOT_EXPERT, ID_RANGE as in foremoe_replication (instance output all -1).
 */
int foremoe_replica_search(const foremoe_shape_t *shape, int32_t M, int32_t max_copies, int64_t a, int64_t b,
                           const int32_t *hist_v, const int32_t *placed_slot_expert_mb,
                           int32_t *slot_expert_mb, int32_t *replicas, int64_t *F, int32_t *dev_status,
                           void *stream);

/* Bytes of device arena foremoe_step_host needs for this shape (includes the assign workspace).
 * mb_off_h: host [n_mb+1] (the arena holds activations of the largest micro-step).  Host only. */
int foremoe_step_host_arena_bytes(const foremoe_shape_t *shape, const int32_t *mb_off_h,
                                  size_t *bytes /* host, out */);

/*
 * The whole path from HOST buffers (end-to-end leg): copies the trace, boundaries and placement
 * to the device, runs load_hist + assign for the step, then for every micro-step i and layer l
 * copies x of the micro-step in (once per micro-step), runs dispatch + combine with the identity
 * expert (expert_out = buf) and copies y back.  Synchronises `stream` before returning.
 *   ids_h [L][T][K], w_h [L][T][K], mb_off_h [n_mb+1], slot_expert_h [L][S]: host (pinned for speed).
 *   x_h   [T][H] host activations (one row per token of the step; reused by every layer).
 *   quota_h [n_mb][L][S], rank_load_h [n_mb][L][P], slot_off_h [n_mb][L][S+1]: host out (may be NULL).
 *   y_h   [T][H] fp32 host out: rows of micro-step i are overwritten by every layer in turn, so
 *         on return it holds the last layer's output; every layer's y crosses the bus.
 *   arena device scratch of foremoe_step_host_arena_bytes() bytes, 256-byte aligned.
 *   status_h host int32 out: the OR of all device fault bits of the step.
 */
int foremoe_step_host(const foremoe_shape_t *shape, const int32_t *ids_h, const float *w_h,
                      const int32_t *mb_off_h, const int32_t *slot_expert_h, const void *x_h,
                      int32_t *quota_h, int32_t *rank_load_h, int32_t *slot_off_h, float *y_h,
                      void *arena, size_t arena_bytes, int32_t *status_h, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* FOREMOE_H_ */
