// fs_kernels.h — host-side launchers of the CUDA kernels behind the C ABI (internal).
// Each launcher enqueues on `st`, returns the number of kernels it launched, and never
// synchronises.  Pointers are device pointers unless stated.
#pragma once

#include "fs_common.cuh"

// Optional per-kernel timing (fs_set_timing): CUDA event pairs recorded on the caller's stream
// around the kernels bench.py reports rooflines for.  NULL = no timing.
enum { FS_T_PLACE_SCORE = 0, FS_T_PLACE_DECODE, FS_T_SUMMARY, FS_T_LOCAL_SLOT, FS_T_LOCAL_SPLIT,
       FS_T_CONSOL_AGG, FS_T_CONSOL_PAIR, FS_T_PLACE_WARM, FS_T_BATCH_TASKS, FS_T_DISPATCH, FS_T_COUNT };
struct FsTimers {
  cudaEvent_t beg[FS_T_COUNT], end[FS_T_COUNT];
  bool used[FS_T_COUNT];
};
static inline void fs_tm_beg(FsTimers* t, int i, cudaStream_t st) { if (t) { cudaEventRecord(t->beg[i], st); } }
static inline void fs_tm_end(FsTimers* t, int i, cudaStream_t st) { if (t) { cudaEventRecord(t->end[i], st); t->used[i] = true; } }

// device-resident view of everything fs_load_profiles / fs_set_gpu_state own
struct FsView {
  FsDimsDev d;
  const float* lat;    // [M][2][F][S][B]
  const float* pow;
  const float2* lpT;   // [M][2][B][S][F]  {LAT, POW}: the plane layout
  const FsPlaneMin* pmin;  // [M][2][B][S]  prefix minima of every plane over shares <= s, all phi
  const fs_model_info* models;
  int K;
  const fs_gpu_state* states;
  const FsGpuInfo* ginfo;   // [K]
  const float* gA;          // [K][FS_NVAR][F]  co-resident energy per variant, INF = infeasible
  const FsGpuRec* grec;     // [Kpad]           compact records, Kpad = K rounded up to FS_CHUNK
  const float* gA0;         // [Kpad][FT]       variant 0 of gA, row stride FT = F rounded up to 32,
                            //                  padding = INF (what the dense kernel stages by TMA)
  int Kpad, FT;
  const FsGpuRec* gsort;    // [Kpad]           grec in the dense kernel's scan order (fs_summary.cu)
  const double* dsuf;       // [Kpad/32 + 3]    [0] magnitude bound, [1+c] suffix minimum of d from chunk c on, [last] earliest T_avail
  int* flag;                // sticky range-error flag (mapped host memory)
};

// fs_tables.cu — validate (finite, > 0) and build the plane layout
int fsk_build_planes(const float* lat, const float* pow, float2* lpT, FsPlaneMin* pmin, FsDimsDev d,
                     int* flag, cudaStream_t st);

// fs_summary.cu — per-GPU co-resident summary: segmented max / slot-order sum
int fsk_summary(const FsView& v, FsGpuInfo* ginfo, float* gA, FsGpuRec* grec, float* gA0, float* okey,
                cudaStream_t st, FsTimers* tm);
int fsk_place_prepare(const FsView& v, const FsGpuRec* grec, FsGpuRec* gsort, double* dsort, double* dsuf,
                      int32_t* warm_off, int32_t* warm_cursor, FsWarmItem* items, cudaStream_t st, FsTimers* tm);

// fs_place.cu — placement scoring + 64-bit-key argmin + decode
struct FsPlaceScratch {
  unsigned long long* keys;        // [R]  (dE, flat) argmin keys
  unsigned long long* stats;       // [8] work counters of the last call: chunks of 32 GPUs tested, cold pairs
                                   // eligible, cold pairs swept, cold candidates swept, warm items tested, pairs
                                   // scored by the definition, candidates scored by the definition, requests
  unsigned int* ctr;               // [nslice <= Kpad/32] dynamic request counters of the dense kernel
  // bucketing of GPUs by model (built by fs_set_gpu_state): warm lists
  const int32_t* warm_off;         // [M+1]
  const FsWarmItem* witems;        // [<= 4K] items, grouped by model
  int sm_count;                    // SMs of the device (grid sizing)
  bool count_work;                 // fill `stats` (fs_set_work_stats): the same kernel with its counters switched on
};
int fsk_place_smem_attr();
int fsk_place(const FsView& v, int R, const fs_request* reqs, fs_placement* out,
              const FsPlaceScratch& sc, cudaStream_t st, FsTimers* tm);
// the paper's three-phase dispatcher at (F_curr, SM_free)
int fsk_dispatch(const FsView& v, int R, const fs_request* reqs, fs_placement* out, const int32_t* warm_off,
                 const FsWarmItem* witems, cudaStream_t st, FsTimers* tm);
int fsk_dispatch_commit(const FsView& v, int R, const fs_request* reqs, fs_placement* out, fs_gpu_avail* work,
                        cudaStream_t st, FsTimers* tm);
// fs_local.cu — per-slot batch search + SM-split search
#define FS_LOCAL_QB 16    // queue-depth buckets per (model, phase) key of the slot search
struct FsLocalScratch {
  float* G;               // [n][RMAX*2][F*S]  slot cost g_{i,p}[phi][sigma]
  const uint32_t* comp;   // [RMAX][ns_stride] SM splits in lexicographic order, sigma_i in byte i
  const uint32_t* comp_n; // [RMAX] number of splits NS = C(S-1, n_res-1)
  int ns_stride;
  // per-call grouping of the live slots by (model, phase, q bucket)
  int32_t* bin_off;       // [M*2*FS_LOCAL_QB + 1]
  int32_t* bin_cursor;    // [M*2*FS_LOCAL_QB]
  int32_t* keylist;       // [M*2] non-empty (model, phase) keys
  int32_t* nkeys;         // [1]
  void* slots;            // [n*8] 16-byte slot records
};
int fsk_local_smem_attr();   // raise the split kernel's dynamic shared memory limit (once)
int fsk_local(const FsView& v, int n, const int32_t* gpu_ids, uint32_t flags, fs_local_cfg* out,
              const FsLocalScratch& sc, cudaStream_t st, FsTimers* tm);

// fs_consol.cu — per-tenant minimum share, per-GPU aggregates, pair scoring
struct FsConsolScratch {
  uint8_t* need;     // [F][K]  sum of minimum shares per frequency, FS_NEED_INF = none
  float* E;          // [F][K]  slot-order energy at those shares
  float2* E2;        // [ceil(F/2)+1][K]  {E[phi], E[phi+1]} per frequency pair (what the pair kernel streams)
  uint32_t* T2;      // [ceil(F/2)+1][K]  S_eff - need of the pair as two binary16 values
  float4* agg;       // [K]     {mem, C*, mig, n_res as float bits}
  unsigned long long* keys;  // [K] per-source argmin key (score, dst)
};
int fsk_consolidate(const FsView& v, const fs_params& prm, fs_consol_out* out,
                    const FsConsolScratch& sc, cudaStream_t st, FsTimers* tm);

// fs_batch.cu — unified priority score + priority batching with bypass
int fsk_batch_tasks(const FsView& v, int n, const int32_t* gpu_ids, const int32_t* off,
                    const fs_task* tasks, fs_task_out* out, int n_tasks, cudaStream_t st, FsTimers* tm);

// fs_alg1.cu — Algorithm 1 phase 1 and the Energy Waste Ratio (first part)
int fsk_llm_profile(const FsView& v, int n, const fs_llm* llms, fs_llm_profile* out, cudaStream_t st);
int fsk_ewr(int n, const int32_t* gpu_of, const float* f_mhz, const float* t_ms, int K, float* fg, double* out3,
            int* flag, cudaStream_t st);

// fs_plan.cu — Algorithm 1 phases 2-3 (sequential part): one warp
size_t fsk_plan_scratch_bytes(int n);
int fsk_replace_plan(int n, const fs_plan_llm* llms, int s_eff, float m_eff, void* scratch, int32_t* gpu_of,
                     int32_t* summary, int* flag, cudaStream_t st);

// fs_migrate.cu — Appendix E: transmission plan (Kuhn-Munkres) and selective migration
int fsk_assign(int n, const float* bytes_mb, const float* bw, int32_t* dst_of, long long* total_us, int* flag,
               cudaStream_t st);
int fsk_migration_select(int r, const fs_mig_req* q, uint8_t* out, float* mig_ms, cudaStream_t st);

#ifdef __CUDACC__
// One co-resident ("tenant") at frequency phi with share sigma, wait = 0 because its slo is the
// REMAINING slack (R:s12).  bump = one more sequence joins its decode batch: the decode bucket
// moves to beta_1+1 when its decode queue is non-empty; past the table -> not ok, e = INF.
// e = fl(e_prefill + e_decode) (Eq. 1); ok = both deadlines hold.
struct TenantE { bool ok; float e; };
__device__ __forceinline__ TenantE tenant_eval(const FsView& v, const fs_tenant& t, int phi,
                                               int sigma, bool bump) {
  const FsDimsDev& d = v.d;
  const int b1 = t.beta[1] + ((bump && t.q[1] > 0) ? 1 : 0);
  TenantE r;
  if (b1 >= d.B) { r.ok = false; r.e = FS_INF; return r; }
  bool ok = true; float e0 = 0.0f, e1 = 0.0f;
  if (t.q[0] > 0) {
    const size_t i = fs_plane(d, t.model, 0, t.beta[0]) + (size_t)sigma * d.F + phi;
    const float2 e = v.lpT[i];
    FsSlot s = fs_slot(0, e.x, e.y, fs_ceil_div(t.q[0], t.beta[0] + 1u), 0.0f, t.slo_ms[0]);
    ok = ok && s.ok; e0 = s.e;
  }
  if (t.q[1] > 0) {
    const size_t i = fs_plane(d, t.model, 1, b1) + (size_t)sigma * d.F + phi;
    const float2 e = v.lpT[i];
    FsSlot s = fs_slot(1, e.x, e.y, fs_ceil_div(t.q[1], b1 + 1u), 0.0f, t.slo_ms[1]);
    ok = ok && s.ok; e1 = s.e;
  }
  r.ok = ok; r.e = __fadd_rn(e0, e1);
  return r;
}
#endif
