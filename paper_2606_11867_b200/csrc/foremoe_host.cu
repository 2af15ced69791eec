// foremoe_step_host: the whole path driven from HOST buffers (the end-to-end leg of the bench and
// the call a host-side user makes).  Orchestration only: every step runs in the kernels behind
// foremoe_plan (= foremoe_load_hist + foremoe_assign) / foremoe_dispatch / foremoe_combine.  Host<->device copies
// run on two side streams so that the x upload of micro-step i+1 and the y download of instance
// n-1 overlap the kernels of instance n.  Contract: include/foremoe.h.
#include "foremoe_common.cuh"

namespace foremoe {

struct Arena {
  size_t ids, w, mb_off, slot_expert, hist, quota, rank_load, slot_off, pair_slot, inv, workspace,
      status, x[2], buf, y[2], total;
};

static Arena make_arena(const Dims &d, size_t max_tokens) {
  Arena a;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += ((bytes + 255) / 256) * 256; return o; };
  const size_t pairs = (size_t)d.L * d.T * d.K;
  a.ids = take(pairs * 4);
  a.w = take(pairs * 4);
  a.mb_off = take(((size_t)d.n_mb + 1) * 4);
  a.slot_expert = take((size_t)d.n_pl * d.S * 4);
  a.hist = take((size_t)d.n_inst * d.E * 4);
  a.quota = take((size_t)d.n_inst * d.S * 4);
  a.rank_load = take((size_t)d.n_inst * d.P * 4);
  a.slot_off = take((size_t)d.n_inst * (d.S + 1) * 4);
  a.pair_slot = take(pairs * 4);
  a.inv = take(pairs * 4);
  a.workspace = take(make_workspace(d).total);
  a.status = take(4);
  a.x[0] = take(max_tokens * d.row_bytes);
  a.x[1] = take(max_tokens * d.row_bytes);
  a.buf = take(max_tokens * d.K * d.row_bytes);
  a.y[0] = take(max_tokens * d.H * 4);
  a.y[1] = take(max_tokens * d.H * 4);
  a.total = off;
  return a;
}

static int check_mb_off_host(const Dims &d, const int32_t *mb_off_h, size_t *max_tokens) {
  if (!mb_off_h || mb_off_h[0] != 0 || mb_off_h[d.n_mb] != d.T) return FOREMOE_ERR_INVALID_ARG;
  size_t mx = 0;
  for (int i = 0; i < d.n_mb; i++) {
    if (mb_off_h[i + 1] < mb_off_h[i]) return FOREMOE_ERR_INVALID_ARG;
    size_t n = (size_t)(mb_off_h[i + 1] - mb_off_h[i]);
    if (n > mx) mx = n;
  }
  *max_tokens = mx;
  return FOREMOE_OK;
}

}  // namespace foremoe

using namespace foremoe;

extern "C" __attribute__((visibility("default"))) int foremoe_step_host_arena_bytes(
    const foremoe_shape_t *shape, const int32_t *mb_off_h, size_t *bytes) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  size_t mx = 0;
  if (!bytes || (rc = check_mb_off_host(d, mb_off_h, &mx))) return FOREMOE_ERR_INVALID_ARG;
  *bytes = make_arena(d, mx).total;
  return FOREMOE_OK;
}

#define FM_CUDA(call) do { if ((call) != cudaSuccess) { rc = FOREMOE_ERR_CUDA; goto done; } } while (0)
#define FM_CALL(call) do { if ((rc = (call)) != FOREMOE_OK) goto done; } while (0)

extern "C" __attribute__((visibility("default"))) int foremoe_step_host(
    const foremoe_shape_t *shape, const int32_t *ids_h, const float *w_h, const int32_t *mb_off_h,
    const int32_t *slot_expert_h, const void *x_h, int32_t *quota_h, int32_t *rank_load_h,
    int32_t *slot_off_h, float *y_h, void *arena, size_t arena_bytes, int32_t *status_h,
    void *stream) {
  Dims d;
  int rc = make_dims(shape, &d);
  if (rc) return rc;
  size_t mx = 0;
  if ((rc = check_mb_off_host(d, mb_off_h, &mx))) return rc;
  if (!ids_h || !w_h || !slot_expert_h || !x_h || !y_h || !arena || !aligned(arena, 256))
    return FOREMOE_ERR_INVALID_ARG;
  const Arena a = make_arena(d, mx);
  if (arena_bytes < a.total) return FOREMOE_ERR_WORKSPACE;

  cudaStream_t st = (cudaStream_t)stream;
  cudaStream_t up = nullptr, down = nullptr;
  cudaEvent_t x_ready[2] = {}, x_free[2] = {}, y_ready[2] = {}, y_free[2] = {}, plan_in = nullptr;
  char *base = (char *)arena;
  int32_t *ids = (int32_t *)(base + a.ids), *mb_off = (int32_t *)(base + a.mb_off);
  float *w = (float *)(base + a.w);
  int32_t *slot_expert = (int32_t *)(base + a.slot_expert), *hist = (int32_t *)(base + a.hist);
  int32_t *quota = (int32_t *)(base + a.quota), *rank_load = (int32_t *)(base + a.rank_load);
  int32_t *slot_off = (int32_t *)(base + a.slot_off), *pair_slot = (int32_t *)(base + a.pair_slot);
  int32_t *inv = (int32_t *)(base + a.inv), *status = (int32_t *)(base + a.status);
  const size_t pairs = (size_t)d.L * d.T * d.K;
  int n_y = 0;

  FM_CUDA(cudaStreamCreateWithFlags(&up, cudaStreamNonBlocking));
  FM_CUDA(cudaStreamCreateWithFlags(&down, cudaStreamNonBlocking));
  for (int b = 0; b < 2; b++) {
    FM_CUDA(cudaEventCreateWithFlags(&x_ready[b], cudaEventDisableTiming));
    FM_CUDA(cudaEventCreateWithFlags(&x_free[b], cudaEventDisableTiming));
    FM_CUDA(cudaEventCreateWithFlags(&y_ready[b], cudaEventDisableTiming));
    FM_CUDA(cudaEventCreateWithFlags(&y_free[b], cudaEventDisableTiming));
  }
  FM_CUDA(cudaEventCreateWithFlags(&plan_in, cudaEventDisableTiming));

  // the side streams start after whatever the caller already queued on `stream`
  FM_CUDA(cudaEventRecord(plan_in, st));
  FM_CUDA(cudaStreamWaitEvent(up, plan_in, 0));
  FM_CUDA(cudaStreamWaitEvent(down, plan_in, 0));

  // plan: trace in, histogram + assignment for the whole step, plan out
  FM_CUDA(cudaMemsetAsync(status, 0, 4, st));
  FM_CUDA(cudaMemcpyAsync(mb_off, mb_off_h, ((size_t)d.n_mb + 1) * 4, cudaMemcpyHostToDevice, st));
  FM_CUDA(cudaMemcpyAsync(slot_expert, slot_expert_h, (size_t)d.n_pl * d.S * 4, cudaMemcpyHostToDevice, st));
  FM_CUDA(cudaMemcpyAsync(ids, ids_h, pairs * 4, cudaMemcpyHostToDevice, st));
  FM_CUDA(cudaMemcpyAsync(w, w_h, pairs * 4, cudaMemcpyHostToDevice, up));   // not needed before combine
  FM_CALL(foremoe_plan(shape, ids, mb_off, slot_expert, nullptr, hist, nullptr, quota, rank_load, slot_off,
                       pair_slot, inv, base + a.workspace, make_workspace(d).total, status, st));
  if (quota_h) FM_CUDA(cudaMemcpyAsync(quota_h, quota, (size_t)d.n_inst * d.S * 4, cudaMemcpyDeviceToHost, st));
  if (rank_load_h) FM_CUDA(cudaMemcpyAsync(rank_load_h, rank_load, (size_t)d.n_inst * d.P * 4, cudaMemcpyDeviceToHost, st));
  if (slot_off_h) FM_CUDA(cudaMemcpyAsync(slot_off_h, slot_off, (size_t)d.n_inst * (d.S + 1) * 4, cudaMemcpyDeviceToHost, st));

  for (int i = 0; i < d.n_mb; i++) {
    const size_t t0 = (size_t)mb_off_h[i], n_tok = (size_t)mb_off_h[i + 1] - t0;
    if (n_tok == 0) continue;
    const int xb = i & 1;
    // upload x of micro-step i once its buffer is no longer read by micro-step i-2
    FM_CUDA(cudaStreamWaitEvent(up, x_free[xb], 0));
    FM_CUDA(cudaMemcpyAsync(base + a.x[xb], (const char *)x_h + t0 * d.row_bytes, n_tok * d.row_bytes,
                            cudaMemcpyHostToDevice, up));
    FM_CUDA(cudaEventRecord(x_ready[xb], up));
    FM_CUDA(cudaStreamWaitEvent(st, x_ready[xb], 0));
    for (int l = 0; l < d.L; l++) {
      const int yb = n_y++ & 1;
      FM_CUDA(cudaStreamWaitEvent(st, y_free[yb], 0));
      FM_CALL(foremoe_dispatch(shape, l, i, i + 1, mb_off, inv, base + a.x[xb], nullptr, base + a.buf, status, st));
      FM_CALL(foremoe_combine(shape, l, i, i + 1, mb_off, inv, w, base + a.buf, (float *)(base + a.y[yb]), status, st));
      FM_CUDA(cudaEventRecord(y_ready[yb], st));
      FM_CUDA(cudaStreamWaitEvent(down, y_ready[yb], 0));
      FM_CUDA(cudaMemcpyAsync(y_h + t0 * d.H, base + a.y[yb], n_tok * d.H * 4, cudaMemcpyDeviceToHost, down));
      FM_CUDA(cudaEventRecord(y_free[yb], down));
    }
    FM_CUDA(cudaEventRecord(x_free[xb], st));
  }
  if (status_h) FM_CUDA(cudaMemcpyAsync(status_h, status, 4, cudaMemcpyDeviceToHost, st));
  FM_CUDA(cudaStreamSynchronize(up));
  FM_CUDA(cudaStreamSynchronize(down));
  FM_CUDA(cudaStreamSynchronize(st));

done:
  if (rc != FOREMOE_OK) cudaDeviceSynchronize();
  for (int b = 0; b < 2; b++) {
    if (x_ready[b]) cudaEventDestroy(x_ready[b]);
    if (x_free[b]) cudaEventDestroy(x_free[b]);
    if (y_ready[b]) cudaEventDestroy(y_ready[b]);
    if (y_free[b]) cudaEventDestroy(y_free[b]);
  }
  if (plan_in) cudaEventDestroy(plan_in);
  if (up) cudaStreamDestroy(up);
  if (down) cudaStreamDestroy(down);
  return rc;
}
