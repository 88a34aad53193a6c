// fs_batch.cu — fs_batch_tasks: steps 1-2 of the local scheduler (§3.4, Fig. 8).
//
// Step 1, unified priority score (Eq. 4):
//   Score = Latency(task) / (Slack - beta*Age),  beta = 0 decode, 1 prefill;
//   Latency(task) = LUT[model][phase][F_curr][sigma][beta_bucket]; used-up slack -> +INF (R:s26).
// Step 2, priority-based task batching: walk the tasks in descending score (ties:
// lowest task index), admit a task iff its SM share and memory still fit, otherwise bypass it.
//
// One block per GPU.  The order is a bitonic sort of 64-bit keys (~orderable(score), index) in
// shared memory; the greedy walk is done by warp 0, 32 sorted tasks at a time: a ballot finds the
// first task that fits what is left, it is admitted, and the search resumes behind it.  The tasks
// it skipped can be dropped for good because the budgets only shrink, so the result is exactly
// the sequential walk's.
#include "fs_kernels.h"

namespace {

constexpr int BT_THREADS = 128;

__device__ __forceinline__ bool task_valid(const fs_task& t, const FsDimsDev& d) {
  return t.model >= 0 && t.model < d.M && t.phase < 2 && t.sigma < d.S && t.beta < d.B;
}

__global__ void __launch_bounds__(BT_THREADS) batch_tasks_kernel(FsView v, int n,
                                                                const int32_t* __restrict__ gpu_ids,
                                                                const int32_t* __restrict__ off,
                                                                const fs_task* __restrict__ tasks,
                                                                fs_task_out* __restrict__ out, int n_tasks) {
  __shared__ unsigned long long skey[FS_MAX_TASKS];
  __shared__ int sbad;
  const FsDimsDev d = v.d;
  const int gi = blockIdx.x;
  const int k = gpu_ids ? gpu_ids[gi] : gi;
  const int t0 = off[gi], t1 = off[gi + 1], nt = t1 - t0;
  if (threadIdx.x == 0) sbad = 0;
  __syncthreads();
  const bool bad_gpu = k < 0 || k >= v.K || t0 < 0 || t1 > n_tasks || nt < 0 || nt > FS_MAX_TASKS;
  int f_cur = 0; float mem_free = 0.0f;
  if (!bad_gpu) { f_cur = v.states[k].f_cur; mem_free = v.states[k].mem_free_mb; }
  const bool bad_f = bad_gpu || f_cur < 0 || f_cur >= d.F;
  if (bad_f) {
    if (!bad_gpu || (t0 >= 0 && t1 <= n_tasks && nt >= 0))
      for (int i = threadIdx.x; i < nt; i += blockDim.x) out[t0 + i] = fs_task_out{0.0f, 0.0f, -1, 0};
    if (threadIdx.x == 0) fs_raise(v.flag, FS_FLAG_ARG);
    return;
  }
  int P = 1;
  while (P < nt) P <<= 1;
  // ---- step 1: scores and sort keys ---------------------------------------------------------
  for (int i = threadIdx.x; i < P; i += blockDim.x) {
    unsigned long long key = FS_KEY_NONE;
    if (i < nt) {
      const fs_task t = tasks[t0 + i];
      if (!task_valid(t, d)) sbad = 1;
      else {
        const float lat = v.lat[fs_idx(d, t.model, t.phase, f_cur, t.sigma, t.beta)];
        const float denom = t.phase == 0 ? __fsub_rn(t.slack_ms, t.age_ms) : t.slack_ms;
        const float score = denom > 0.0f ? __fdiv_rn(lat, denom) : FS_INF;
        out[t0 + i].score = score; out[t0 + i].latency_ms = lat;
        key = ((unsigned long long)(~fs_orderable(score)) << 32) | (uint32_t)i;   // descending score
      }
    }
    skey[i] = key;
  }
  __syncthreads();
  if (sbad) {
    for (int i = threadIdx.x; i < nt; i += blockDim.x) out[t0 + i] = fs_task_out{0.0f, 0.0f, -1, 0};
    if (threadIdx.x == 0) fs_raise(v.flag, FS_FLAG_ARG);
    return;
  }
  // ---- bitonic sort, ascending keys -----------------------------------------------------------
  for (int size = 2; size <= P; size <<= 1)
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = threadIdx.x; i < (P >> 1); i += blockDim.x) {
        const int lo = ((i / stride) * stride << 1) + (i % stride), hi = lo + stride;
        const bool up = (lo & size) == 0;
        const unsigned long long a = skey[lo], b = skey[hi];
        if ((a > b) == up) { skey[lo] = b; skey[hi] = a; }
      }
      __syncthreads();
    }
  // ---- step 2: greedy admission in score order (warp 0) ---------------------------------------
  if (threadIdx.x >= 32) return;
  const int lane = threadIdx.x;
  int sm_left = d.S; float mem_left = mem_free;
  for (int base = 0; base < nt; base += 32) {
    const int pos = base + lane;
    int idx = 0, need = 0x7FFFFFFF; float mem = FS_INF;
    if (pos < nt) {
      idx = (int)(uint32_t)skey[pos];
      const fs_task t = tasks[t0 + idx];
      need = (int)t.sigma + 1; mem = t.mem_mb;
    }
    bool adm = false; int cur = 0;
    for (;;) {
      const unsigned fit = __ballot_sync(0xffffffffu, lane >= cur && need <= sm_left && mem <= mem_left);
      if (fit == 0u) break;
      const int j = __ffs(fit) - 1;
      if (lane == j) adm = true;
      sm_left -= __shfl_sync(0xffffffffu, need, j);
      mem_left = __fsub_rn(mem_left, __shfl_sync(0xffffffffu, mem, j));
      cur = j + 1;
    }
    if (pos < nt) { out[t0 + idx].rank = pos; out[t0 + idx].admitted = adm ? 1 : 0; }
  }
}

}  // namespace

int fsk_batch_tasks(const FsView& v, int n, const int32_t* gpu_ids, const int32_t* off,
                    const fs_task* tasks, fs_task_out* out, int n_tasks, cudaStream_t st, FsTimers* tm) {
  if (n <= 0) return 0;
  fs_tm_beg(tm, FS_T_BATCH_TASKS, st);
  batch_tasks_kernel<<<n, BT_THREADS, 0, st>>>(v, n, gpu_ids, off, tasks, out, n_tasks);
  fs_tm_end(tm, FS_T_BATCH_TASKS, st);
  return 1;
}
