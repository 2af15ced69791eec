// Shared device/host helpers of the ForeMoE sm_100a library (internal; the public contract is
// include/foremoe.h).  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/foremoe.h"

namespace foremoe {

constexpr int kChunkPairs = 4096;    // pairs ranked by one CTA of k_assign_pairs / k_chunk_hist
#ifndef FOREMOE_CHUNK_THREADS
#define FOREMOE_CHUNK_THREADS 256
#endif
constexpr int kChunkThreads = FOREMOE_CHUNK_THREADS;
constexpr int kChunkWarps = kChunkThreads / 32;
constexpr int kRankShift = 20;       // k_assign_pairs packs (expert id, rank inside the warp's segment) into one int
static_assert(kChunkPairs / kChunkWarps <= (1 << (31 - kRankShift)), "rank inside a warp's segment must fit");
constexpr int kQuotaThreads = 128;
constexpr int kMaxWaterPasses = 256;  // Phase B cap (O2)

// Derived sizes, computed once per call on the host.
struct Dims {
  int L, E, K, P, Nb, Nr, Ns, S, T, n_mb, H, act_dtype;
  int es;            // bytes per activation element
  int row_bytes;     // H * es
  int row_vec;       // row_bytes / 16
  int n_inst;        // n_mb * L
  int n_pl;          // number of placements: L or n_mb * L
  int pl_per_mb;     // 1 if one placement per micro-step
  int plan_stable;   // FOREMOE_FLAG_PLAN_STABLE: plan arrays may be read before the grid-dependency wait
  int tpc;           // tokens per chunk
  int max_chunks;    // upper bound on chunks per layer
};

inline int make_dims(const foremoe_shape_t *s, Dims *d) {
  if (!s) return FOREMOE_ERR_INVALID_ARG;
  if (s->L <= 0 || s->E <= 0 || s->K <= 0 || s->P <= 0 || s->Nb <= 0 || s->Nr < 0 || s->T < 0 ||
      s->n_mb <= 0 || s->H <= 0)
    return FOREMOE_ERR_INVALID_ARG;
  if (s->K > s->E || s->K > 32) return FOREMOE_ERR_INVALID_ARG;
  if (s->E % s->P != 0 || s->Nb != s->E / s->P) return FOREMOE_ERR_INVALID_ARG;
  if (s->act_dtype != FOREMOE_ACT_BF16 && s->act_dtype != FOREMOE_ACT_FP32)
    return FOREMOE_ERR_INVALID_ARG;
  if ((int64_t)s->T * s->K >= ((int64_t)1 << 31)) return FOREMOE_ERR_INVALID_ARG;
  d->L = s->L; d->E = s->E; d->K = s->K; d->P = s->P; d->Nb = s->Nb; d->Nr = s->Nr;
  d->Ns = s->Nb + s->Nr;
  if ((int64_t)d->P * d->Ns >= ((int64_t)1 << 24)) return FOREMOE_ERR_INVALID_ARG;
  d->S = d->P * d->Ns;
  d->T = s->T; d->n_mb = s->n_mb; d->H = s->H; d->act_dtype = s->act_dtype;
  d->es = s->act_dtype == FOREMOE_ACT_BF16 ? 2 : 4;
  int64_t rb = (int64_t)s->H * d->es;
  if (rb % 16 != 0 || rb >= ((int64_t)1 << 30)) return FOREMOE_ERR_INVALID_ARG;
  d->row_bytes = (int)rb;
  d->row_vec = (int)(rb / 16);
  if ((int64_t)s->n_mb * s->L >= ((int64_t)1 << 28)) return FOREMOE_ERR_INVALID_ARG;
  d->n_inst = s->n_mb * s->L;
  if (s->placement_mb_stride == 0) { d->n_pl = s->L; d->pl_per_mb = 0; }
  else if (s->placement_mb_stride == s->L * d->S) { d->n_pl = d->n_inst; d->pl_per_mb = 1; }
  else return FOREMOE_ERR_INVALID_ARG;
  if (s->flags & ~FOREMOE_FLAG_PLAN_STABLE) return FOREMOE_ERR_INVALID_ARG;
  d->plan_stable = (s->flags & FOREMOE_FLAG_PLAN_STABLE) ? 1 : 0;
  d->tpc = kChunkPairs / s->K;
  d->max_chunks = (s->T + d->tpc - 1) / d->tpc + s->n_mb;
  return FOREMOE_OK;
}

inline bool aligned(const void *p, size_t a) { return ((uintptr_t)p % a) == 0; }

// Workspace carve-up of foremoe_assign (all sections int32, 16-byte aligned).
struct Workspace {
  size_t chunk_off, mb_ok, pl_host_ptr, pl_host_slot, pl_active, pl_rslot, pl_fault, inst_cum_end,
      inst_slot_adj, inst_ok, chunk_cnt, total;
};

inline Workspace make_workspace(const Dims &d) {
  Workspace w;
  size_t off = 0;
  auto take = [&](size_t n_int) { size_t o = off; off += ((n_int * 4 + 15) / 16) * 16; return o; };
  w.chunk_off = take((size_t)d.n_mb + 1);
  w.mb_ok = take(4);
  w.pl_host_ptr = take((size_t)d.n_pl * (d.E + 1));
  w.pl_host_slot = take((size_t)d.n_pl * d.S);
  w.pl_active = take((size_t)d.n_pl * d.S);
  w.pl_rslot = take((size_t)d.n_pl * d.S);
  w.pl_fault = take((size_t)d.n_pl);
  w.inst_cum_end = take((size_t)d.n_inst * d.S);
  w.inst_slot_adj = take((size_t)d.n_inst * d.S);
  w.inst_ok = take((size_t)d.n_inst);
  w.chunk_cnt = take((size_t)d.L * d.max_chunks * d.E);
  w.total = off;
  return w;
}

__device__ __forceinline__ void raise_fault(int32_t *dev_status, int bits) {
  if (dev_status && bits) atomicOr(dev_status, bits);
}

// Largest i in [0, n) with off[i] <= v, for a non-decreasing off[0..n] with off[0] <= v < off[n]:
// the last of any run of equal boundaries, so empty ranges are skipped.
__device__ __forceinline__ int find_range(const int32_t *__restrict__ off, int n, int v) {
  int lo = 0, hi = n;          // invariant: off[lo] <= v < off[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (__ldg(off + mid) <= v) lo = mid; else hi = mid;
  }
  return lo;
}

int num_sms();

// The launchers memoise per-kernel launch facts (SM count, occupancy, the opt-in shared-memory
// attribute).  They are per DEVICE and must be safe when several host threads drive several
// streams or devices at once, so a memo is a small table of atomics indexed by the calling
// thread's current device: a slot holds 0 (unknown) or (key << 16 | value).  Two threads that miss
// at the same time compute the same fact twice and store the same word: no lock is needed.
constexpr int kMaxDevices = 64;
constexpr int kMemoWays = 4;

inline int current_device() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return -1;
  return dev;
}

struct DeviceMemo {
  std::atomic<uint64_t> slot[kMaxDevices][kMemoWays];
  // The keys of one memo differ in their high bits (shared-memory bytes * 2048 + threads, threads a
  // multiple of 32), so the way is taken from a multiplicative hash of the key, not from its low bits;
  // a key lives in the first free way at or after its home way, and get() looks at all of them.  Only
  // a fifth distinct key per device and kernel instantiation evicts (its home way).
  static_assert(kMemoWays == 4, "home() returns the top two bits of the hash");
  static unsigned home(uint64_t key) { return (unsigned)((key * 0x9E3779B97F4A7C15ull) >> 62); }
  // value in [1, 65535] or 0 when (dev, key) is not cached; key < 2^47
  int get(int dev, uint64_t key) const {
    if (dev < 0) return 0;
    const unsigned h = home(key);
    for (unsigned i = 0; i < (unsigned)kMemoWays; i++) {
      const uint64_t v = slot[dev][(h + i) % kMemoWays].load(std::memory_order_acquire);
      if ((v >> 16) == key + 1) return (int)(v & 0xffff);
    }
    return 0;
  }
  void put(int dev, uint64_t key, int value) {
    if (dev < 0 || value <= 0 || value > 0xffff) return;
    const uint64_t word = ((key + 1) << 16) | (uint64_t)value;
    const unsigned h = home(key);
    for (unsigned i = 0; i < (unsigned)kMemoWays; i++) {
      std::atomic<uint64_t> &s = slot[dev][(h + i) % kMemoWays];
      uint64_t v = s.load(std::memory_order_acquire);
      if ((v >> 16) == key + 1) return;                                  // another thread was first: same fact
      if (v == 0 && s.compare_exchange_strong(v, word, std::memory_order_acq_rel)) return;
      if ((v >> 16) == key + 1) return;                                  // lost the race to the same key
    }
    slot[dev][h].store(word, std::memory_order_release);               // all ways taken by other keys
  }
};

}  // namespace foremoe
