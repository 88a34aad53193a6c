// fs_migrate.cu — Appendix E: the transmission plan and the selective-migration rules.
//
// fs_migration_plan: e_uv = Bytes(u -> v) / BW(u, v) in whole microseconds,
//   c_uv = rint(fl(fl(bytes_u / bw_uv) * 1000)), minimum-cost assignment by the Kuhn-Munkres algorithm in
//   its shortest-augmenting-path form with row / column potentials (exact in int64; ties: lowest column).
//   The n augmentations are sequential; inside one, the scan over the columns (reduced costs, running
//   minima, the next column) and the potential update are lane <-> column.  One warp, state in shared
//   memory (n <= 1024).
// fs_migration_select: per in-flight request, KV transfer iff faster than recomputation; migrate iff the
//   remaining computation on the source exceeds the migration time.
#include "fs_kernels.h"

namespace {

constexpr int MG_MAXN = 1024;
constexpr long long MG_BIG = 1ll << 60;

__device__ __forceinline__ long long mg_cost(const float* bytes_mb, const float* bw, int n, int u, int v) {
  return __float2ll_rn(__fmul_rn(__fdiv_rn(bytes_mb[u], bw[(size_t)u * n + v]), 1000.0f));
}

__global__ void __launch_bounds__(32) assign_kernel(int n, const float* __restrict__ bytes_mb, const float* __restrict__ bw,
                                                   int32_t* __restrict__ dst_of, long long* __restrict__ total_us, int* flag) {
  __shared__ long long pu[MG_MAXN + 1], pv[MG_MAXN + 1], minv[MG_MAXN + 1];
  __shared__ int p[MG_MAXN + 1], way[MG_MAXN + 1];
  __shared__ unsigned char used[MG_MAXN + 1];
  const int lane = threadIdx.x;
  bool bad = false;
  for (int x = lane; x < n * n; x += 32) bad = bad || !(bw[x] > 0.0f && bw[x] < FS_INF);
  for (int u = lane; u < n; u += 32) bad = bad || !(bytes_mb[u] >= 0.0f && bytes_mb[u] < FS_INF);
  if (__any_sync(0xffffffffu, bad) && lane == 0) fs_raise(flag, FS_FLAG_ARG);
  for (int j = lane; j <= n; j += 32) { pu[j] = 0; pv[j] = 0; p[j] = 0; way[j] = 0; }
  __syncwarp();
  for (int i = 1; i <= n; ++i) {
    for (int j = lane; j <= n; j += 32) { minv[j] = MG_BIG; used[j] = 0; }
    if (lane == 0) p[0] = i;
    __syncwarp();
    int j0 = 0;
    do {
      if (lane == 0) used[j0] = 1;
      __syncwarp();
      const int i0 = p[j0];
      const long long pui = pu[i0];
      long long delta = MG_BIG; int j1 = 0;
      for (int j = 1 + lane; j <= n; j += 32) {
        if (used[j]) continue;
        const long long cur = mg_cost(bytes_mb, bw, n, i0 - 1, j - 1) - pui - pv[j];
        long long mv = minv[j];
        if (cur < mv) { mv = cur; minv[j] = cur; way[j] = j0; }
        if (mv < delta) { delta = mv; j1 = j; }        // ascending j per lane: strict < keeps the lowest
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const long long od = __shfl_xor_sync(0xffffffffu, delta, o);
        const int oj = __shfl_xor_sync(0xffffffffu, j1, o);
        if (od < delta || (od == delta && oj != 0 && (j1 == 0 || oj < j1))) { delta = od; j1 = oj; }
      }
      __syncwarp();
      for (int j = lane; j <= n; j += 32) {
        if (used[j]) { pu[p[j]] += delta; pv[j] -= delta; } else minv[j] -= delta;
      }
      j0 = j1;
      __syncwarp();
    } while (p[j0] != 0);
    if (lane == 0) {
      int j = j0;
      do { const int jn = way[j]; p[j] = p[jn]; j = jn; } while (j);
    }
    __syncwarp();
  }
  for (int j = 1 + lane; j <= n; j += 32) dst_of[p[j] - 1] = j - 1;
  __syncwarp();
  long long tot = 0;
  for (int u = lane; u < n; u += 32) tot += mg_cost(bytes_mb, bw, n, u, dst_of[u]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
  if (lane == 0) *total_us = tot;
}

__global__ void migration_select_kernel(int r, const fs_mig_req* __restrict__ q, uint8_t* __restrict__ out,
                                        float* __restrict__ mig_ms) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= r) return;
  const fs_mig_req x = q[i];
  const float kv_tx = __fdiv_rn(x.kv_mb, x.bw_mb_per_ms);
  const bool kv = kv_tx < x.recompute_ms;
  const float t = __fadd_rn(__fdiv_rn(x.tokens_mb, x.bw_mb_per_ms), kv ? kv_tx : x.recompute_ms);
  mig_ms[i] = t;
  out[i] = (uint8_t)((x.remaining_ms > t ? 1 : 0) | (kv ? 2 : 0));
}

}  // namespace

int fsk_assign(int n, const float* bytes_mb, const float* bw, int32_t* dst_of, long long* total_us, int* flag,
               cudaStream_t st) {
  assign_kernel<<<1, 32, 0, st>>>(n, bytes_mb, bw, dst_of, total_us, flag);
  return 1;
}

int fsk_migration_select(int r, const fs_mig_req* q, uint8_t* out, float* mig_ms, cudaStream_t st) {
  if (r <= 0) return 0;
  migration_select_kernel<<<(r + 255) / 256, 256, 0, st>>>(r, q, out, mig_ms);
  return 1;
}
