/* festina_eval.h — C ABI of libfestina_eval (sm_100a CUDA implementation).
 *
 * The batched, SLO-constrained energy argmin of Festina's control plane
 * (arxiv/paper_2606_30391): global placement (§3.3, Eq. 2-3), per-GPU local
 * configuration (§3.4, Fig. 8 step 3) and GPU x GPU consolidation scoring (§3.5).
 * "P:NNN" cites a line of the paper text; "R:sNN" cites a reading listed in
 * DESIGN.md ("Readings of the paper").
 *
 * Conventions common to every call
 *   - Plain C types only.  Every bulk pointer of one call lives in the memory space named by
 *     `space` (FS_HOST: ordinary or pinned host memory, FS_DEVICE: device memory of the
 *     context's CUDA device).  Small descriptor structs (fs_dims, fs_params) are always host.
 *   - The caller owns all in/out buffers.  Inputs are COPIED into context-owned device memory;
 *     the caller may reuse them once `cuda_stream` has passed the call (FS_HOST inputs that are
 *     not pinned are consumed before the call returns).  Outputs are written into the caller's
 *     buffer; FS_HOST outputs are valid after the call returns, FS_DEVICE outputs after the
 *     caller synchronises `cuda_stream`.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Return value: FS_OK (0) or a negative fs_status.  Nothing throws or aborts across the ABI.
 *     Host-visible arguments are validated synchronously.  Device-resident data are
 *     range-checked inside the kernels; a violation sets a sticky flag that the NEXT call
 *     returns (and clears) as FS_ERR_RANGE.  FS_HOST calls wait for their own kernels and report their own
 *     flags; for FS_DEVICE / FS_HOST_PINNED calls the flag is reported by the first later call on the context
 *     (whichever it is): FS_ERR_RANGE then says that SOME earlier asynchronous call saw bad data, and the
 *     records it affected carry gpu / phi / dst = -1.
 *   - No feasible candidate: index fields are -1 and the value field is +INF
 *     (the caller's cue to scale out).
 *   - All arithmetic is IEEE-754 binary32, round-to-nearest-even, no FMA contraction, in the
 *     bracketing DESIGN.md states; integer quantities are exact.
 *   - One context per host thread; calls on one context are not re-entrant.  Calls that do not depend on
 *     each other's outputs (fs_place_batch / fs_dispatch vs fs_local_config vs fs_consolidate, all after
 *     fs_set_gpu_state) may be issued on different streams by that thread; the caller orders the streams.
 *     fs_place_batch, fs_dispatch and fs_dispatch_commit share staging buffers: one of them at a time.
 *   - FS_DEVICE and FS_HOST_PINNED calls never synchronise and do not allocate once a call of the same sizes has run, so a
 *     sequence of them can be captured into a CUDA graph (with fs_set_timing off) and replayed.  The scan order
 *     and the per-model lists of the placement calls are built by the FIRST fs_place_batch / fs_dispatch after
 *     an fs_set_gpu_state: capture fs_set_gpu_state in the same graph as the placement calls that follow it (a
 *     graph holding only a placement call would replay against the lists of the state it was captured with).
 *   - There is no CPU fallback: every entry point runs CUDA kernels on the context's device.
 */
#ifndef FESTINA_EVAL_H
#define FESTINA_EVAL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fs_ctx fs_ctx; /* opaque: device copies of tables/state + scratch */

typedef enum {
  FS_OK = 0,
  FS_ERR_ARG = -1,   /* NULL pointer, bad enum, bad count                       */
  FS_ERR_SHAPE = -2, /* dims outside the supported range                        */
  FS_ERR_STATE = -3, /* call order: profiles / GPU state not loaded yet; or a call that has to allocate
                        (first call of these sizes) was made while `cuda_stream` is being captured: run
                        it once outside the capture first                                          */
  FS_ERR_RANGE = -4, /* an index / value inside device data was out of range    */
  FS_ERR_CUDA = -5,  /* a CUDA runtime call failed (see fs_last_cuda_error)     */
  FS_ERR_NOMEM = -6  /* device or host allocation failed                        */
} fs_status;

enum {
  FS_HOST = 0,        /* host memory; the call returns when the outputs are in the caller's buffer          */
  FS_DEVICE = 1,      /* device memory; the call returns after enqueueing its work on `cuda_stream`          */
  FS_HOST_PINNED = 2  /* page-locked host memory, asynchronous: copies and kernels are enqueued on
                         `cuda_stream` and the call returns without waiting.  Inputs must stay untouched and
                         outputs are valid only after the caller synchronises the stream; range flags
                         surface on the next call (as with FS_DEVICE).  fs_place_batch reads the requests and
                         writes the records in place over PCIe when the buffers are mapped into the device's
                         address space (cudaHostAlloc / cudaHostRegister; otherwise, or with FS_ZERO_COPY=0
                         in the environment, by bulk copies).  Accepted by the calls of the serving
                         loop: fs_set_gpu_state, fs_place_batch, fs_local_config, fs_consolidate, fs_dispatch;
                         the others return FS_ERR_ARG.                                                       */
};

/* flags of fs_local_config: one objective bit and one split-mode bit (R:s8, R:s9) */
enum {
  FS_OBJ_ENERGY = 0,       /* slot cost = energy  t*POW ("lowest predicted energy") */
  FS_OBJ_POWER = 1,        /* slot cost = power   POW   ("minimize power")           */
  FS_SPLIT_EXHAUSTIVE = 0, /* all SM splits with sum == S                                  */
  FS_SPLIT_MINSM = 2       /* per-task minimum SM, sum <= S (Fig. 8 step 3)         */
};

#define FS_RMAX 4   /* tenant slots per GPU (co-resident models)            */
#define FS_PHASES 2 /* 0 = prefill (TTFT), 1 = decode (TBT) */

/* Limits checked by fs_load_profiles (FS_ERR_SHAPE otherwise). */
#define FS_MAX_M 32767
#define FS_MAX_F 256
#define FS_MAX_S 32
#define FS_MAX_B 256

/* Table axes: M models, F frequency levels (ascending MHz), S SM-share levels
 * (index sigma <-> share (sigma+1)/S), B batch levels (index beta <-> batch beta+1).   */
typedef struct { int32_t M, F, S, B; } fs_dims;

/* Per model: weight-load (cold start) latency P:177; KV-cache MB per token (R:s13);
 * weight footprint; energy of migrating the model.                              */
typedef struct { float load_ms, kv_mb_per_token, weights_mb, mig_mj; } fs_model_info;

/* Consolidation constants: idle power, horizon Delta, per-GPU memory
 * capacity, safety margin delta in percent.                                      */
typedef struct { float p_idle_w, horizon_ms, mem_cap_mb; int32_t delta_pct; } fs_params;

/* One co-resident model ("tenant") of a GPU: its model id, its SM share index sigma
 * (share = sigma+1 units), per phase the batch bucket beta, queued tokens q and the
 * REMAINING SLO slack in ms (slo_ms[0] TTFT-like, slo_ms[1] TBT), and its memory use.    */
typedef struct {
  int16_t model; uint8_t sigma, _p0;
  uint8_t beta[2], _p1[2];
  uint32_t q[2];
  float slo_ms[2];
  float mem_used_mb;
} fs_tenant; /* 28 bytes */

/* Per-GPU state summary: number of tenants (0 = inactive GPU, never a
 * candidate), current frequency index F_curr, earliest-available time T_avail, free memory. */
typedef struct {
  int32_t n_res, f_cur;
  float t_avail_ms, mem_free_mb;
  fs_tenant t[FS_RMAX];
} fs_gpu_state; /* 128 bytes, 16-byte aligned */

/* Request descriptor: model, prompt length L = Req_in, PREDICTED output length
 * o_pred (the 5 % pad is applied inside), TTFT and TBT SLOs in ms, caller tag (echoed
 * nowhere; free for the caller).                                                         */
typedef struct {
  int32_t model; uint32_t L, o_pred;
  float slo_ttft_ms, slo_tbt_ms;
  uint32_t tag, _pad[2];
} fs_request; /* 32 bytes */

/* Placement decision: GPU, granted share index sigma, frequency index phi, decode batch
 * bucket beta the request joins, f_req = lowest feasible frequency index at (gpu, sigma),
 * marginal energy Delta-E in mJ, TTFT and TBT estimates, flat = (gpu*S + sigma)*F + phi.  */
typedef struct {
  int32_t gpu; int16_t sigma, phi, beta, f_req;
  float energy_mj, ttft_ms, tbt_ms;
  uint32_t flat, _pad;
} fs_placement; /* 32 bytes */

/* Local configuration of one GPU: frequency, per tenant share index and per slot batch
 * bucket, objective value, energy and power at the choice.                               */
typedef struct {
  int16_t phi, f_req;
  uint8_t sigma[FS_RMAX];
  uint8_t beta[FS_RMAX][2];
  float cost, energy_mj, power_w;
  uint32_t flat, _pad[4];
} fs_local_cfg; /* 48 bytes */

/* Consolidation result per source GPU: best destination, frequency index of the merged
 * GPU, extra energy the destination pays, net saving of draining the source.             */
typedef struct { int32_t dst, phi; float score_mj, saving_mj; } fs_consol_out; /* 16 bytes */

/* One active LLM for Algorithm 1, phase 1: its model, the average input / output length of
 * the last window, its SLOs and its measured request arrival rate (requests per second).  32 bytes. */
typedef struct {
  int32_t model; uint32_t avg_in, avg_out; float slo_ttft_ms, slo_tbt_ms, lambda_rps; uint32_t _pad[2];
} fs_llm;
/* (sigma_p, phi_p), (sigma_d, phi_d): energy-optimal feasible LUT configuration of the prefill / decode
 * phase, with its duration t_*_ms and power p_*_w; sm_units = Eq. 8 in share units, need_units =
 * ceil(sm_units) = l.S; phi_l = l.F, the energy-optimal feasible frequency at l.S units, t_l_ms and
 * e_l_mj the LLM's time and energy there; mem_mb = M_l by Little's law.  -1 / +INF where a
 * phase (or l.F) has no feasible configuration.  48 bytes.                                      */
typedef struct {
  int16_t sigma_p, phi_p, sigma_d, phi_d; float t_p_ms, t_d_ms, p_p_w, p_d_w;
  float sm_units; int16_t need_units, phi_l; float t_l_ms, e_l_mj, mem_mb; uint32_t _pad;
} fs_llm_profile;

/* LLM descriptor of Algorithm 1: l.S = need_units (share units, >= 1), l.M = mem_mb,
 * l.F = f_mhz (preferred frequency), t_ms = its execution time (the weight of Eq. 5).  16 bytes. */
typedef struct { int32_t need_units; float mem_mb, f_mhz, t_ms; } fs_plan_llm;

/* What the commit pass of fs_dispatch_commit changes in a GPU's record: 16 bytes. */
typedef struct { float t_avail_ms, mem_free_mb; int32_t f_cur; uint32_t _pad; } fs_gpu_avail;

/* One in-flight request at reconfiguration time: remaining computation on the source,
 * token state and KV-cache size, the bandwidth of its source -> destination link under the chosen
 * mapping, and the time to recompute its KV cache on the destination.  32 bytes.               */
typedef struct { float remaining_ms, tokens_mb, kv_mb, bw_mb_per_ms, recompute_ms; uint32_t _pad[3]; } fs_mig_req;
#define FS_MIG_MIGRATE 1u   /* else: finish on the source */
#define FS_MIG_KV 2u        /* transfer the KV cache; else tokens only and recompute */

/* One runnable task of the local scheduler's priority queue (Fig. 8 steps 1-2): a
 * decode step or a prefill unit of `model`, run with `sigma`+1 SM share units at batch bucket
 * `beta`.  slack_ms = remaining time to its SLO deadline (TBT for decode, TTFT for prefill),
 * age_ms = time since it became runnable, mem_mb = memory it needs while running.  24 bytes. */
typedef struct {
  int16_t model; uint8_t phase, sigma, beta, _p0[3];
  float slack_ms, age_ms, mem_mb; uint32_t tag;
} fs_task;
/* score = Eq. 4 (+INF when the effective slack is used up), latency_ms = the LUT entry it used,
 * rank = position in descending-score order (ties: lowest index), admitted = 1 if the greedy
 * walk put it into the batch.  rank = -1: the GPU's task list was rejected (FS_ERR_RANGE). 16 bytes. */
typedef struct { float score, latency_ms; int32_t rank, admitted; } fs_task_out;
#define FS_MAX_TASKS 1024  /* tasks per GPU in one fs_batch_tasks call */

/* Create / destroy a context bound to CUDA device `cuda_device`.
 * fs_create: *out receives the context; FS_ERR_CUDA if the device cannot be used.        */
int fs_create(fs_ctx** out, int cuda_device);
int fs_destroy(fs_ctx* ctx);

/* fs_load_profiles — the offline look-up table (§3.2.1; axes R:s1).
 *   lat, pow : [M][2][F][S][B] fp32, row-major, beta fastest; latency in ms, power in W;
 *              every entry finite and > 0.
 *   freq_mhz : [F] ascending (informational; the arithmetic uses indices only).
 *   models   : [M];  params: host struct.
 * The library keeps its own copies (and a second, (sigma,phi)-plane-contiguous layout
 * [M][2][B][S][F] built on the device).  Replaces any previously loaded profiles and
 * invalidates the GPU state.  Errors: FS_ERR_ARG, FS_ERR_SHAPE, FS_ERR_NOMEM, FS_ERR_CUDA. */
int fs_load_profiles(fs_ctx* ctx, const fs_dims* dims, const float* lat, const float* pow,
                     const float* freq_mhz, const fs_model_info* models,
                     const fs_params* params, int space, void* cuda_stream);

/* fs_set_gpu_state — the per-GPU state summaries the global scheduler polls.
 *   states : [K] records.  Invariants (FS_ERR_RANGE on the next call if violated; such a GPU
 *            is treated as inactive): 0 <= n_res <= 4, model/sigma/beta/f_cur in range,
 *            sum(sigma_i+1) <= S, q < 2^24.
 * Launches the summary kernel: per GPU, per frequency and per "one more sequence on tenant j"
 * variant, co-resident feasibility (the segmented max over co-residents)
 * and the slot-order energy sum.                                     */
int fs_set_gpu_state(fs_ctx* ctx, int32_t K, const fs_gpu_state* states, int space,
                     void* cuda_stream);

/* fs_place_batch — global dispatch (§3.3; Eq. 2-3; R:s2-s6).
 * Every request is scored against the same state snapshot over all (GPU k, grant sigma,
 * frequency phi); out[r] is the feasible candidate minimising (Delta-E, flat).
 *   reqs : [R];  out : [R].  R = 0 is a no-op.                                            */
int fs_place_batch(fs_ctx* ctx, int32_t R, const fs_request* reqs, fs_placement* out,
                   int space, void* cuda_stream);

/* fs_local_config — per-GPU runtime resource allocation (§3.4, Fig. 8 step 3).
 *   n, gpu_ids : the GPUs to configure; gpu_ids == NULL means GPUs 0..n-1 (n <= K).
 *   flags      : FS_OBJ_* | FS_SPLIT_*.
 *   out        : [n].                                                                      */
int fs_local_config(fs_ctx* ctx, int32_t n, const int32_t* gpu_ids, uint32_t flags,
                    fs_local_cfg* out, int space, void* cuda_stream);

/* fs_consolidate — drain-one-source scoring over all GPU pairs (§3.5; margin
 * P:351; idle power vs migration energy P:46; R:s17-s20).   out : [K].             */
int fs_consolidate(fs_ctx* ctx, fs_consol_out* out, int space, void* cuda_stream);

/* The paper's own dispatcher (Fig. 6): one operating point per GPU, S_k = SM_free and
 * f_k = F_curr.  Phase 1: feasibility of the request at F_curr (same eligibility as
 * fs_place_batch).  Phase 2: E^k = Power x Latency of the request's own work (Eq. 2), argmin
 * (Eq. 3); among GPUs within 2 % of the minimum the most free memory wins, then the largest
 * SM_free, then the lowest index.  Phase 3: if none is feasible, the first GPU in
 * ascending T_avail that is feasible at F_max (last frequency level); else scale-out: gpu = -1
 * and sigma = S-1, phi = the energy-optimal feasible frequency of a fresh GPU (wait = load_ms).
 * Output records as fs_place_batch, except: energy_mj = E^k (not a marginal energy) and f_req =
 * the phase that decided (1 = F_curr, 2 = F_max retry, 3 = scale-out, -1 = infeasible even on
 * a fresh GPU).  Requires K < 2^24.  reqs : [R]; out : [R]; both in `space`.                  */
int fs_dispatch(fs_ctx* ctx, int32_t R, const fs_request* reqs, fs_placement* out, int space,
                void* cuda_stream);

/* fs_dispatch with the sequential commit pass between the requests of one batch (
 * R:s34 of P:214-218).  The requests are dispatched in the order given, each against the records the
 * previous ones left.  A request sent to GPU k in phase 1 or 2 starts at its wait time with all of
 * SM_free_k and holds it until it completes:
 *   T_avail_k  <- fl(ttft + fl(ceil(O/(beta+1)) * tbt))   (its completion: when the next one can start)
 *   mem_free_k <- fl(mem_free_k - Req_mem)                 (reserved until the next poll)
 *   F_curr_k   <- phi                                       (the F_max retry leaves the GPU at F_max)
 * Scale-out decisions (gpu = -1) change nothing; the resident models stay those of fs_set_gpu_state.
 * The context's own GPU state is NOT modified: `after` ([K], may be NULL) receives the three fields of
 * every GPU after the last commit; the caller feeds the next poll through fs_set_gpu_state.
 * One thread block (a cluster of up to 8 for 2,049..16,384 GPUs) walks the requests (they are serial by
 * definition); the GPUs are the parallel axis.
 *   reqs : [R]; out : [R]; after : [K] or NULL; all in `space`.  Requires K < 2^24.              */
int fs_dispatch_commit(fs_ctx* ctx, int32_t R, const fs_request* reqs, fs_placement* out,
                       fs_gpu_avail* after, int space, void* cuda_stream);

/* Local scheduler steps 1-2 for n GPUs (Eq. 4, Fig. 8): unified priority
 * score of every runnable task at the GPU's current frequency, then priority-based batching with
 * bypass under the budgets "all S share units" and the GPU's free memory (fs_set_gpu_state).
 * gpu_ids : [n] or NULL (= GPUs 0..n-1);  task_off : [n+1], tasks of entry i are
 * tasks[task_off[i] .. task_off[i+1]) (at most FS_MAX_TASKS each);  tasks, out : [n_tasks].
 * All bulk pointers live in `space`.  Invalid ids / fields raise FS_ERR_RANGE (sticky) and mark
 * that GPU's outputs with rank = -1.                                                           */
int fs_batch_tasks(fs_ctx* ctx, int32_t n, const int32_t* gpu_ids, const int32_t* task_off,
                   const fs_task* tasks, fs_task_out* out, int32_t n_tasks, int space,
                   void* cuda_stream);

/* Algorithm 1, phase 1 (Eq. 8, Little's law) for n active LLMs: see
 * fs_llm_profile.  Needs fs_load_profiles only.  llms, out : [n], in `space`.                   */
int fs_llm_profiles(fs_ctx* ctx, int32_t n, const fs_llm* llms, fs_llm_profile* out, int space,
                    void* cuda_stream);

/* Energy Waste Ratio (Eq. 5-7) of a placement of n LLMs on K GPUs: gpu_of[l] = GPU of LLM l
 * (< 0: not placed), f_mhz[l] = its preferred frequency F_l, t_ms[l] = its execution time t_l.
 * f_gpu[g] = F_g = the highest F_l on GPU g (0 if empty); out3 = {E_waste, E_optimal, EWR} in
 * binary64 (sums over the LLMs; EWR = 0 when E_optimal = 0).  All pointers in `space`.           */
int fs_ewr(fs_ctx* ctx, int32_t n, const int32_t* gpu_of, const float* f_mhz, const float* t_ms,
           int32_t K, float* f_gpu, double* out3, int space, void* cuda_stream);

/* Algorithm 1, phases 2-3 for n active LLMs against the effective capacities
 * s_eff (share units) and m_eff (MB) of one GPU ((1 - delta) of the real ones).
 * Phase 2: summary[0] = N_sm, summary[1] = N_mem (Best-Fit-Decreasing bin counts), summary[2] =
 * N_min = their maximum.  Phase 3: the LLMs in ascending f_mhz go to the GPU with the closest
 * operating frequency (the highest f_mhz on it; an empty GPU is the last resort) if they fit;
 * else the target's lowest-frequency resident moves to the second-closest GPU when that is
 * resource-valid and lowers the waste of Eq. 5; else the second-closest GPU; else the closest other GPU
 * that fits; else a new GPU.  gpu_of[l] = the GPU of LLM l (-1: it exceeds a whole GPU);
 * summary[3] = GPUs in use or planned (>= N_min).  Ties: lower index everywhere.
 * llms : [n]; gpu_of : [n]; summary : [4]; all in `space`.  need_units < 1 raises FS_ERR_RANGE.   */
int fs_replace_plan(fs_ctx* ctx, int32_t n, const fs_plan_llm* llms, int32_t s_eff, float m_eff,
                    int32_t* gpu_of, int32_t* summary, int space, void* cuda_stream);

/* fs_replace_plan for callers that must not allocate device memory.
 *
 * Everything else in this header hangs off an fs_ctx, and a context allocates: fs_create does, and so does
 * the first call of each size.  That rules the library out for two kinds of caller.  One is a scheduler that
 * sits next to a serving engine which claimed almost all of HBM for weights and KV cache when it started:
 * a cudaMalloc issued later may simply fail.  The other is a control loop sharing the GPU with live
 * inference: cudaMalloc and cudaFree serialise on the driver's allocator, and cudaFree waits for the whole
 * device, so either one stalls the streams the scheduler is supposed to leave alone.  This call is for them.
 * It takes no context and calls no cudaMalloc / cudaFree / cudaHostAlloc nor any routine that allocates; the
 * kernel's working arrays sit in one array compiled into the library (about 300 KiB), which every GPU that
 * loads the library keeps until the process exits.  That fixed size is the limit:
 *   n <= FS_PLAN_STATIC_MAX_N, otherwise FS_ERR_SHAPE ("dims outside the supported range") and nothing runs.
 *
 * Same kernel, same results as fs_replace_plan(..., FS_DEVICE, ...):
 *   llms [n], gpu_of [n], summary [4] : caller-owned memory the CURRENT CUDA device can address (device
 *   memory, or mapped page-locked host memory); the work is enqueued on `cuda_stream`, which must belong
 *   to the current device, and the call returns without waiting.  s_eff in 1..FS_MAX_S (else FS_ERR_ARG).
 *   An LLM with need_units < 1 stays unplaced (gpu_of = -1) as in fs_replace_plan, but with no context there
 *   is nowhere to keep the sticky FS_ERR_RANGE: check that field yourself if it can be bad.
 * First call on each device: the library looks up the array's device address (one cudaGetSymbolAddress,
 * which also makes the runtime load the library's code on that device).  Make that first call early, at
 * start-up, and before any stream capture begins on that device.
 * The array is shared by every call in the process.  Nothing in it needs clearing between calls (the kernel
 * writes each word before reading it), but two calls that overlap on one GPU - different streams, or
 * different host threads - race on it: keep them on one stream, or order the streams yourself.
 * Errors: FS_ERR_ARG, FS_ERR_SHAPE, FS_ERR_CUDA (no usable device, or the launch failed).                */
#define FS_PLAN_STATIC_MAX_N 1024
int fs_replace_plan_static(int32_t n, const fs_plan_llm* llms, int32_t s_eff, float m_eff,
                           int32_t* gpu_of, int32_t* summary, void* cuda_stream);

/* Transmission plan: minimum-cost assignment of n sources to n destinations under
 * e_uv = Bytes(u -> v) / BW(u, v), costs in whole microseconds rint(fl(fl(bytes_mb[u] / bw[u][v]) * 1000))
 * (bytes in MB, bw in MB per ms, row-major [n][n], > 0), Kuhn-Munkres, exact in int64.
 * dst_of[u] = destination of source u; *total_us = the minimum total cost.  n <= 1024.           */
int fs_migration_plan(fs_ctx* ctx, int32_t n, const float* bytes_mb, const float* bw_mb_per_ms,
                      int32_t* dst_of, int64_t* total_us, int space, void* cuda_stream);
/* Selective request migration for r in-flight requests: flags[i] = FS_MIG_KV if sending the
 * KV cache (kv_mb / bw) is faster than recomputing it, | FS_MIG_MIGRATE if the remaining computation on
 * the source exceeds the migration time mig_ms[i] = tokens_mb / bw + min-option above.          */
int fs_migration_select(fs_ctx* ctx, int32_t r, const fs_mig_req* reqs, uint8_t* flags, float* mig_ms,
                        int space, void* cuda_stream);

/* Diagnostics. */
const char* fs_strerror(int code);
int fs_last_cuda_error(const fs_ctx* ctx); /* cudaError_t of the last failed runtime call */
/* Kernels launched by this context since creation (bench.py's gpu_launches counter).     */
uint64_t fs_launch_count(const fs_ctx* ctx);
/* Work counters of fs_place_batch (measurement only).  fs_set_work_stats(ctx, 1) makes later
 * fs_place_batch calls run the scoring kernel with its work counters switched on (same kernel, same
 * results, a little slower); fs_last_place_stats copies the counters of the most recent such call
 * (it synchronises the device):
 *   out[0] chunks of 32 GPU records tested (lane <-> GPU: eligibility + lower bound)
 *   out[1] cold (request, GPU) pairs found eligible      out[2] cold pairs swept after pruning
 *   out[3] cold candidates swept (sum of sm_free*F)      out[4] warm (model resident) pairs tested
 *   out[5] pairs scored candidate by candidate with the definition (warm pairs + tie recovery)
 *   out[6] candidates scored that way                    out[7] requests processed (x GPU slices)
 *   out[8] requests for which the (sigma, phi) tile was built (a cold pair could still win)        */
#define FS_NSTATS 9
int fs_set_work_stats(fs_ctx* ctx, int on);
int fs_last_place_stats(fs_ctx* ctx, uint64_t out[FS_NSTATS]);

/* Per-kernel device timing for measurement (bench.py's roofline line).  fs_set_timing(ctx, 1)
 * makes every later call record CUDA event pairs on its stream around its kernels;
 * fs_get_timing waits for them and writes the duration in ms of the MOST RECENT launch of each
 * timed kernel into ms[0..n) (-1 = never launched), indexed by fs_timer.                    */
typedef enum {
  FS_TIMER_PLACE_SCORE = 0, /* fs_place_batch: dense candidate scoring + argmin       */
  FS_TIMER_PLACE_DECODE,    /* key -> fs_placement                                   */
  FS_TIMER_SUMMARY,         /* co-resident summary of fs_set_gpu_state               */
  FS_TIMER_LOCAL_SLOT,      /* per-slot batch search of fs_local_config              */
  FS_TIMER_LOCAL_SPLIT,     /* SM-split search of fs_local_config                    */
  FS_TIMER_CONSOL_AGG,      /* per-tenant minimum shares of fs_consolidate           */
  FS_TIMER_CONSOL_PAIR,     /* pair scoring of fs_consolidate                        */
  FS_TIMER_PLACE_WARM,      /* scan order + warm lists, built by the first placement call after fs_set_gpu_state */
  FS_TIMER_BATCH_TASKS,     /* fs_batch_tasks: priority score + batching            */
  FS_TIMER_DISPATCH,        /* fs_dispatch: the paper's three-phase dispatcher      */
  FS_TIMER_COUNT
} fs_timer;
int fs_set_timing(fs_ctx* ctx, int on);
int fs_get_timing(fs_ctx* ctx, float* ms, int n);

#ifdef __cplusplus
}
#endif
#endif /* FESTINA_EVAL_H */
