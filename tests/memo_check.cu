// Host-only check of the launch-fact memo (paper_2606_11867_b200/csrc/foremoe_common.cuh), built and run by
// tests/test_abi.py without a GPU.  Keys as the launchers form them: smem * 2048 + threads, threads a
// multiple of 32 -- all congruent modulo the number of ways.
#include <stdio.h>

#include "../paper_2606_11867_b200/csrc/foremoe_common.cuh"

int main() {
  static foremoe::DeviceMemo memo;
  const uint64_t keys[5] = {(uint64_t)14336 * 2048 + 512, (uint64_t)12288 * 2048 + 512, (uint64_t)66 * 1024 * 2048 + 64,
                            (uint64_t)200 * 1024 * 2048 + 256, (uint64_t)4096 * 2048 + 128};
  for (int dev = 0; dev < 2; dev++) {
    for (int k = 0; k < 4; k++) {
      if (memo.get(dev, keys[k]) != 0) { printf("key %d cached before put\n", k); return 1; }
      memo.put(dev, keys[k], 10 * dev + k + 1);
    }
    for (int k = 0; k < 4; k++)               // four shapes of one instantiation stay cached together
      if (memo.get(dev, keys[k]) != 10 * dev + k + 1) { printf("dev %d key %d evicted\n", dev, k); return 1; }
    memo.put(dev, keys[1], 99);               // a second put of a cached key changes nothing
    if (memo.get(dev, keys[1]) != 10 * dev + 2) { printf("re-put overwrote\n"); return 1; }
  }
  memo.put(0, keys[4], 77);                   // a fifth key evicts exactly one of the four
  int alive = 0;
  for (int k = 0; k < 4; k++) alive += memo.get(0, keys[k]) == k + 1;
  if (memo.get(0, keys[4]) != 77 || alive != 3) { printf("fifth key: alive %d\n", alive); return 1; }
  if (memo.get(-1, keys[0]) != 0 || memo.get(1, keys[4]) != 0) { printf("wrong device hit\n"); return 1; }
  printf("memo ok\n");
  return 0;
}
