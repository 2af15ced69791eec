/*
 * The boundary used from plain C: a caller that knows nothing but include/foremoe.h and the CUDA
 * runtime API.  Plans a tiny step with foremoe_plan, dispatches and combines every instance, and
 * checks on the host what holds for any correct implementation (BASELINE.json north_star):
 *   - histogram sums equal T_i * K, quotas of an expert's slots sum to its count (Eq.(8)),
 *   - inv is a bijection onto the instance's rows and perm is its inverse,
 *   - every gathered row is the bit copy of its token's row,
 *   - combine(dispatch(x)) with weights that sum to 1 per token reproduces x (fp32, exact here: the
 *     weights are 1/2 + 1/2 and x holds small integers).
 * Built and run by tests/test_gpu_c_abi.py (gcc, linked against libforemoe.so and libcudart).
 * Exit code 0 = all checks passed; otherwise the failing check is printed.
 */
#include <cuda_runtime_api.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "foremoe.h"

#define CHECK(c) do { if (!(c)) { fprintf(stderr, "FAILED %s:%d: %s\n", __FILE__, __LINE__, #c); return 1; } } while (0)
#define CU(c) CHECK((c) == cudaSuccess)
#define FM(c) CHECK((c) == FOREMOE_OK)

enum { L = 2, E = 8, K = 2, P = 4, NB = 2, NR = 1, NS = NB + NR, S = P * NS, NMB = 3, H = 64, T = 777 };
static const int32_t mb_off_h[NMB + 1] = {0, 300, 300, 777};        /* one empty micro-step */

static void *dev_copy(const void *h, size_t n) {
  void *d = NULL;
  if (cudaMalloc(&d, n ? n : 16) != cudaSuccess) return NULL;
  if (h && cudaMemcpy(d, h, n, cudaMemcpyHostToDevice) != cudaSuccess) return NULL;
  return d;
}

int main(void) {
  foremoe_shape_t s;
  memset(&s, 0, sizeof s);
  s.L = L; s.E = E; s.K = K; s.P = P; s.Nb = NB; s.Nr = NR; s.T = T; s.n_mb = NMB; s.H = H;
  s.act_dtype = FOREMOE_ACT_FP32;
  CHECK(foremoe_version() >= 200);

  /* trace: skewed ids (two distinct experts per token), weights 1/2 + 1/2 */
  static int32_t ids[L][T][K];
  static float w[L][T][K], x[T][H];
  unsigned r = 12345u;
  for (int l = 0; l < L; l++)
    for (int t = 0; t < T; t++) {
      r = r * 1664525u + 1013904223u;
      int a = (int)((r >> 8) % E);
      if ((r >> 20) % 3 == 0) a = l;                                   /* a hot expert per layer */
      r = r * 1664525u + 1013904223u;
      int b = (a + 1 + (int)((r >> 8) % (E - 1))) % E;
      ids[l][t][0] = a; ids[l][t][1] = b;
      w[l][t][0] = 0.5f; w[l][t][1] = 0.5f;
    }
  for (int t = 0; t < T; t++)
    for (int h = 0; h < H; h++) x[t][h] = (float)((t * 31 + h * 7) % 201 - 100);
  /* placement: rank p holds experts 2p, 2p+1; its replica slot holds the layer's hot expert */
  static int32_t se[L][S];
  for (int l = 0; l < L; l++)
    for (int p = 0; p < P; p++) {
      se[l][p * NS + 0] = 2 * p; se[l][p * NS + 1] = 2 * p + 1;
      se[l][p * NS + 2] = (l / NB == p) ? -1 : l;                       /* not on the rank that already hosts it */
    }

  size_t ws_bytes = 0;
  FM(foremoe_workspace_bytes(&s, &ws_bytes));
  int32_t *d_ids = dev_copy(ids, sizeof ids), *d_mb = dev_copy(mb_off_h, sizeof mb_off_h), *d_se = dev_copy(se, sizeof se);
  float *d_w = dev_copy(w, sizeof w);
  int32_t *d_hist = dev_copy(NULL, sizeof(int32_t) * NMB * L * E), *d_quota = dev_copy(NULL, sizeof(int32_t) * NMB * L * S);
  int32_t *d_rl = dev_copy(NULL, sizeof(int32_t) * NMB * L * P), *d_so = dev_copy(NULL, sizeof(int32_t) * NMB * L * (S + 1));
  int32_t *d_ps = dev_copy(NULL, sizeof ids), *d_inv = dev_copy(NULL, sizeof ids);
  int64_t *d_step = dev_copy(NULL, sizeof(int64_t) * L * E);
  void *d_ws = dev_copy(NULL, ws_bytes);
  int32_t zero = 0, *d_status = dev_copy(&zero, 4);
  CHECK(d_ids && d_mb && d_se && d_w && d_hist && d_quota && d_rl && d_so && d_ps && d_inv && d_step && d_ws && d_status);

  FM(foremoe_plan(&s, d_ids, d_mb, d_se, NULL, d_hist, d_step, d_quota, d_rl, d_so, d_ps, d_inv, d_ws, ws_bytes,
                  d_status, NULL));
  static int32_t hist[NMB][L][E], quota[NMB][L][S], rl[NMB][L][P], inv[L][T][K], ps[L][T][K];
  int32_t status = -1;
  CU(cudaMemcpy(hist, d_hist, sizeof hist, cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(quota, d_quota, sizeof quota, cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(rl, d_rl, sizeof rl, cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(inv, d_inv, sizeof inv, cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(ps, d_ps, sizeof ps, cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(&status, d_status, 4, cudaMemcpyDeviceToHost));
  CHECK(status == 0);

  for (int i = 0; i < NMB; i++)
    for (int l = 0; l < L; l++) {
      const int n_tok = mb_off_h[i + 1] - mb_off_h[i];
      long sum = 0, load = 0;
      for (int e = 0; e < E; e++) {
        sum += hist[i][l][e];
        long q = 0;
        for (int j = 0; j < S; j++)
          if (se[l][j] == e) q += quota[i][l][j];
        CHECK(q == hist[i][l][e]);                                    /* Eq.(8) */
      }
      CHECK(sum == (long)n_tok * K);
      for (int p = 0; p < P; p++) load += rl[i][l][p];
      CHECK(load == (long)n_tok * K);
    }

  /* data path, one instance at a time */
  float *d_x = dev_copy(NULL, sizeof x), *d_buf = dev_copy(NULL, sizeof(float) * T * K * H), *d_y = dev_copy(NULL, sizeof x);
  int32_t *d_perm = dev_copy(NULL, sizeof(int32_t) * T * K);
  static float buf[T * K][H], y[T][H];
  static int32_t perm[T * K];
  static char seen[T * K];
  CHECK(d_x && d_buf && d_y && d_perm);
  for (int l = 0; l < L; l++)
    for (int i = 0; i < NMB; i++) {
      const int t0 = mb_off_h[i], n = mb_off_h[i + 1] - t0;
      CU(cudaMemcpy(d_x, x[t0], sizeof(float) * n * H, cudaMemcpyHostToDevice));
      FM(foremoe_dispatch(&s, l, i, i + 1, d_mb, d_inv, d_x, d_perm, d_buf, d_status, NULL));
      FM(foremoe_combine(&s, l, i, i + 1, d_mb, d_inv, d_w, d_buf, d_y, d_status, NULL));
      CU(cudaDeviceSynchronize());
      CU(cudaMemcpy(buf, d_buf, sizeof(float) * n * K * H, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(perm, d_perm, sizeof(int32_t) * n * K, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(y, d_y, sizeof(float) * n * H, cudaMemcpyDeviceToHost));
      memset(seen, 0, sizeof seen);
      for (int t = 0; t < n; t++)
        for (int k = 0; k < K; k++) {
          const int p = (t0 + t) * K + k, d = inv[l][t0 + t][k] - t0 * K;   /* row inside the instance */
          CHECK(d >= 0 && d < n * K && !seen[d]);
          seen[d] = 1;
          CHECK(perm[d] == p);
          CHECK(se[l][ps[l][t0 + t][k]] == ids[l][t0 + t][k]);          /* the slot hosts the pair's expert, Eq.(9) */
          CHECK(memcmp(buf[d], x[t0 + t], sizeof(float) * H) == 0);
        }
      for (int t = 0; t < n; t++) CHECK(memcmp(y[t], x[t0 + t], sizeof(float) * H) == 0);
    }
  CU(cudaMemcpy(&status, d_status, 4, cudaMemcpyDeviceToHost));
  CHECK(status == 0);
  printf("c_abi_demo ok\n");
  return 0;
}
