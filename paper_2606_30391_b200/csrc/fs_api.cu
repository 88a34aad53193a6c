// fs_api.cu — the C ABI of libfestina_eval (include/festina_eval.h): context, argument
// validation, device-memory ownership, host<->device staging, kernel sequencing.
// No arithmetic of the method lives here (kernels: fs_tables/fs_summary/fs_place/fs_local/
// fs_consol .cu) and there is no CPU fallback: without a CUDA device every call fails.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "fs_kernels.h"

struct fs_ctx {
  int dev = 0;
  fs_dims d{0, 0, 0, 0};
  fs_params prm{0, 0, 0, 0};
  bool have_prof = false, have_state = false, place_ready = false;
  // profiles
  float *lat = nullptr, *pow = nullptr, *freq = nullptr; float2* lpT = nullptr; FsPlaneMin* pmin = nullptr; size_t pmin_cap = 0;
  fs_model_info* models = nullptr;
  size_t table_cap = 0; int m_cap = 0, f_cap = 0;
  uint32_t *comp = nullptr, *comp_n = nullptr; int ns_stride = 1; size_t comp_cap = 0;
  // state + summaries
  int K = 0, k_cap = 0;
  fs_gpu_state* states = nullptr; FsGpuInfo* ginfo = nullptr; float* gA = nullptr; size_t gA_cap = 0;
  FsGpuRec* grec = nullptr; FsGpuRec* gsort = nullptr; double *dsort = nullptr, *dsuf = nullptr; float* gA0 = nullptr; size_t gA0_cap = 0; int Kpad = 0, FT = 32;
  int32_t *warm_off = nullptr, *warm_cursor = nullptr; FsWarmItem* warm_item = nullptr; int warm_m_cap = 0;
  // placement scratch
  int r_cap = 0; unsigned long long* keys = nullptr; unsigned long long* stats = nullptr;
  unsigned int* ctr = nullptr;
  fs_request* reqs_dev = nullptr; fs_placement* place_dev = nullptr;
  // local scratch
  size_t local_cap = 0; int n_cap = 0; float* G = nullptr;
  int32_t* ids_dev = nullptr; fs_local_cfg* local_dev = nullptr;
  int32_t *bin_off = nullptr, *bin_cursor = nullptr, *keylist = nullptr, *nkeys = nullptr; int bin_m_cap = 0;
  uint4* lslots = nullptr;
  // task batching scratch (FS_HOST staging)
  int bt_n_cap = 0, bt_t_cap = 0; int32_t *bt_ids = nullptr, *bt_off = nullptr; fs_task* bt_tasks = nullptr; fs_task_out* bt_out = nullptr;
  // Algorithm 1 / EWR scratch (FS_HOST staging)
  bool zero_copy = true;   // FS_ZERO_COPY=0 in the environment: bulk copies for FS_HOST_PINNED too
  size_t a1_cap = 0; unsigned char* a1_buf = nullptr; size_t pl_cap = 0; unsigned char* pl_buf = nullptr;
  // consolidation scratch
  size_t consol_cap = 0; uint8_t* need = nullptr; float* E = nullptr; float2* E2 = nullptr; uint32_t* T2 = nullptr; float4* agg = nullptr;
  unsigned long long* ckeys = nullptr; fs_consol_out* consol_dev = nullptr;
  // diagnostics
  int* flag_host = nullptr; int* flag_dev = nullptr;
  uint64_t launches = 0; int last_cuda = 0;
  bool timing = false; bool have_events = false; FsTimers tm{};
  int sm_count = 148; bool count_work = false;
  cudaStream_t cur = nullptr;   // the stream of the API call in progress (grow() asks whether it is being captured)
};

namespace {

#define FS_CUDA(ctx, expr)                                   \
  do {                                                       \
    cudaError_t e_ = (expr);                                 \
    if (e_ != cudaSuccess) {                                 \
      (ctx)->last_cuda = (int)e_;                            \
      cudaGetLastError();                                    \
      return e_ == cudaErrorMemoryAllocation ? FS_ERR_NOMEM : FS_ERR_CUDA; \
    }                                                        \
  } while (0)

// The new buffer is allocated before the old one is released: after a failed allocation the pointer and the
// caller's capacity field still describe a valid (old) buffer, and the next call simply tries again.
// A call that has to grow a buffer allocates and (when it replaces one) waits for the device: neither is legal
// while the caller's stream is being captured into a graph, and the synchronisation would silently invalidate the
// capture.  Such a call returns FS_ERR_STATE instead ("run the call once with these sizes before capturing").
template <class T> int grow(fs_ctx* c, T*& p, size_t n_elems) {
  if (n_elems == 0) n_elems = 1;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(c->cur, &cap) != cudaSuccess) { cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
  if (cap != cudaStreamCaptureStatusNone) return FS_ERR_STATE;
  T* fresh = nullptr;
  FS_CUDA(c, cudaMalloc((void**)&fresh, n_elems * sizeof(T)));
  if (p) {
    // kernels of earlier calls may still read the old buffer on the caller's streams
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaFree(p);
    if (e != cudaSuccess) {                 // keep the old buffer (still described by the caller's capacity field)
      cudaFree(fresh);
      c->last_cuda = (int)e; cudaGetLastError();
      return FS_ERR_CUDA;
    }
  }
  p = fresh;
  return FS_OK;
}
#define FS_TRY(x) do { int r_ = (x); if (r_ != FS_OK) return r_; } while (0)

// sticky device-side range errors of earlier calls: report once, then clear
int take_flags(fs_ctx* c) {
  // one atomic exchange per word: a flag a running kernel raises is either seen by this call or left for the
  // next one, never lost between a read and a clear.  (A flag is reported by the first call that sees it, which
  // for FS_DEVICE / FS_HOST_PINNED calls is a later call than the one that caused it: festina_eval.h.)
  int any = 0;
  for (int i = 0; i < FS_NFLAGS; ++i) any |= __atomic_exchange_n(&c->flag_host[i], 0, __ATOMIC_ACQ_REL);
  return any ? FS_ERR_RANGE : FS_OK;
}

int check_kernel(fs_ctx* c) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { c->last_cuda = (int)e; return FS_ERR_CUDA; }
  return FS_OK;
}

FsView view_of(const fs_ctx* c) {
  FsView v;
  v.d = FsDimsDev{c->d.M, c->d.F, c->d.S, c->d.B};
  v.lat = c->lat; v.pow = c->pow; v.lpT = c->lpT; v.pmin = c->pmin; v.models = c->models;
  v.K = c->K; v.states = c->states; v.ginfo = c->ginfo; v.gA = c->gA; v.flag = c->flag_dev;
  v.grec = c->grec; v.gA0 = c->gA0; v.Kpad = c->Kpad; v.FT = c->FT; v.gsort = c->gsort; v.dsuf = c->dsuf;
  return v;
}

// all SM splits of S share units into n positive parts, lexicographic, sigma_0 most significant
void build_splits(int S, std::vector<uint32_t>& comp, uint32_t comp_n[FS_RMAX], int& stride) {
  std::vector<uint32_t> lists[FS_RMAX];
  for (int n = 1; n <= FS_RMAX; ++n) {
    int sg[FS_RMAX] = {0, 0, 0, 0};
    // odometer over (sigma_0..sigma_{n-1}) in lexicographic order, keep sum(sigma_i+1) == S
    while (true) {
      int tot = 0;
      for (int i = 0; i < n; ++i) tot += sg[i] + 1;
      if (tot == S) {
        uint32_t pk = 0;
        for (int i = 0; i < n; ++i) pk |= (uint32_t)sg[i] << (8 * i);
        lists[n - 1].push_back(pk);
      }
      int i = n - 1;
      while (i >= 0 && ++sg[i] >= S) { sg[i] = 0; --i; }
      if (i < 0) break;
    }
    comp_n[n - 1] = (uint32_t)lists[n - 1].size();
  }
  stride = 1;
  for (int n = 0; n < FS_RMAX; ++n) if ((int)comp_n[n] > stride) stride = (int)comp_n[n];
  comp.assign((size_t)stride * FS_RMAX, 0u);
  for (int n = 0; n < FS_RMAX; ++n)
    for (size_t r = 0; r < lists[n].size(); ++r) comp[(size_t)n * stride + r] = lists[n][r];
}

// scan order + warm lists of the placement kernels: once per fs_set_gpu_state, on first use
int place_prepare(fs_ctx* c, cudaStream_t st) {
  if (c->place_ready || c->K <= 0) return FS_OK;
  c->launches += fsk_place_prepare(view_of(c), c->grec, c->gsort, c->dsort, c->dsuf, c->warm_off, c->warm_cursor,
                                   c->warm_item, st, c->timing ? &c->tm : nullptr);
  FS_TRY(check_kernel(c));
  c->place_ready = true;
  return FS_OK;
}

cudaMemcpyKind in_kind(int space) { return space != FS_DEVICE ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice; }
// the calls of the serving loop also take page-locked host buffers without waiting for the stream
bool space_ok(int space) { return space == FS_HOST || space == FS_DEVICE || space == FS_HOST_PINNED; }

}  // namespace

extern "C" {

int fs_create(fs_ctx** out, int cuda_device) {
  if (!out) return FS_ERR_ARG;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) {
    cudaGetLastError();
    return FS_ERR_CUDA;   // no CUDA device: there is no CPU fallback
  }
  fs_ctx* c = new (std::nothrow) fs_ctx();
  if (!c) return FS_ERR_NOMEM;
  c->dev = cuda_device;
  if (cudaSetDevice(cuda_device) != cudaSuccess ||
      cudaHostAlloc((void**)&c->flag_host, sizeof(int) * FS_NFLAGS, cudaHostAllocMapped) != cudaSuccess ||
      cudaHostGetDevicePointer((void**)&c->flag_dev, c->flag_host, 0) != cudaSuccess ||
      cudaMalloc((void**)&c->stats, FS_NSTATS * sizeof(unsigned long long)) != cudaSuccess) {
    cudaGetLastError();
    delete c;
    return FS_ERR_CUDA;
  }
  std::memset(c->flag_host, 0, sizeof(int) * FS_NFLAGS);
  cudaMemset(c->stats, 0, FS_NSTATS * sizeof(unsigned long long));
  fsk_local_smem_attr();
  fsk_place_smem_attr();
  cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, cuda_device);
  if (const char* e = getenv("FS_ZERO_COPY")) c->zero_copy = e[0] != '0';
  *out = c;
  return FS_OK;
}

int fs_destroy(fs_ctx* c) {
  if (!c) return FS_ERR_ARG;
  cudaSetDevice(c->dev);
  cudaDeviceSynchronize();
  void* ptrs[] = {c->lat, c->pow, c->lpT, c->pmin, c->freq, c->models, c->comp, c->comp_n, c->states,
                  c->ginfo, c->gA, c->grec, c->gsort, c->dsort, c->dsuf, c->gA0, c->ctr, c->warm_off, c->warm_cursor, c->warm_item, c->keys, c->stats,
                  c->reqs_dev, c->place_dev, c->bin_off, c->bin_cursor, c->keylist, c->nkeys, c->lslots, c->G, c->ids_dev, c->local_dev, c->need, c->E,
                  c->agg, c->E2, c->T2, c->ckeys, c->consol_dev, c->bt_ids, c->bt_off, c->bt_tasks, c->bt_out, c->a1_buf, c->pl_buf};
  bool ok = true;
  for (void* p : ptrs) if (p) ok = (cudaFree(p) == cudaSuccess) && ok;
  if (c->flag_host) ok = (cudaFreeHost(c->flag_host) == cudaSuccess) && ok;
  if (c->have_events)
    for (int i = 0; i < FS_T_COUNT; ++i) {
      ok = (cudaEventDestroy(c->tm.beg[i]) == cudaSuccess) && ok; ok = (cudaEventDestroy(c->tm.end[i]) == cudaSuccess) && ok;
    }
  cudaGetLastError();
  delete c;
  return ok ? FS_OK : FS_ERR_CUDA;
}

int fs_load_profiles(fs_ctx* c, const fs_dims* dims, const float* lat, const float* pow,
                     const float* freq_mhz, const fs_model_info* models, const fs_params* params,
                     int space, void* cuda_stream) {
  if (!c || !dims || !lat || !pow || !freq_mhz || !models || !params) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  if (dims->M < 1 || dims->M > FS_MAX_M || dims->F < 1 || dims->F > FS_MAX_F || dims->S < 1 ||
      dims->S > FS_MAX_S || dims->B < 1 || dims->B > FS_MAX_B)
    return FS_ERR_SHAPE;
  if (params->delta_pct < 0 || params->delta_pct > 100) return FS_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  c->have_prof = false; c->have_state = false; c->K = 0; c->consol_cap = 0;
  const size_t n = (size_t)dims->M * 2 * dims->F * dims->S * dims->B;
  if (n > c->table_cap) {
    FS_TRY(grow(c, c->lat, n)); FS_TRY(grow(c, c->pow, n));
    FS_TRY(grow(c, c->lpT, n));
    c->table_cap = n;
  }
  if (dims->M > c->m_cap) { FS_TRY(grow(c, c->models, (size_t)dims->M)); c->m_cap = dims->M; }
  if (dims->F > c->f_cap) { FS_TRY(grow(c, c->freq, (size_t)dims->F)); c->f_cap = dims->F; }
  const cudaMemcpyKind kind = in_kind(space);
  FS_CUDA(c, cudaMemcpyAsync(c->lat, lat, n * sizeof(float), kind, st));
  FS_CUDA(c, cudaMemcpyAsync(c->pow, pow, n * sizeof(float), kind, st));
  FS_CUDA(c, cudaMemcpyAsync(c->freq, freq_mhz, dims->F * sizeof(float), kind, st));
  FS_CUDA(c, cudaMemcpyAsync(c->models, models, dims->M * sizeof(fs_model_info), kind, st));
  c->d = *dims; c->prm = *params;
  // SM-split enumeration table of fs_local_config (index bookkeeping only)
  std::vector<uint32_t> comp; uint32_t comp_n[FS_RMAX]; int stride = 1;
  build_splits(dims->S, comp, comp_n, stride);
  if (comp.size() > c->comp_cap) { FS_TRY(grow(c, c->comp, comp.size())); c->comp_cap = comp.size(); }
  if (!c->comp_n) FS_TRY(grow(c, c->comp_n, (size_t)FS_RMAX));
  // synchronous copies: `comp` is a local that dies at return
  FS_CUDA(c, cudaMemcpyAsync(c->comp, comp.data(), comp.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
  FS_CUDA(c, cudaMemcpyAsync(c->comp_n, comp_n, sizeof(comp_n), cudaMemcpyHostToDevice, st));
  FS_CUDA(c, cudaStreamSynchronize(st));
  c->ns_stride = stride;
  { const size_t nd = (size_t)dims->M * 2 * dims->B * dims->S;
    if (nd > c->pmin_cap) { FS_TRY(grow(c, c->pmin, nd)); c->pmin_cap = nd; } }
  c->launches += fsk_build_planes(c->lat, c->pow, c->lpT, c->pmin,
                                  FsDimsDev{dims->M, dims->F, dims->S, dims->B}, c->flag_dev, st);
  FS_TRY(check_kernel(c));
  c->have_prof = true;
  return pending;
}

int fs_set_gpu_state(fs_ctx* c, int32_t K, const fs_gpu_state* states, int space, void* cuda_stream) {
  if (!c || K < 0 || (K > 0 && !states)) return FS_ERR_ARG;
  if (!space_ok(space)) return FS_ERR_ARG;
  if (!c->have_prof) return FS_ERR_STATE;
  if ((unsigned long long)K * c->d.S * c->d.F >= 0xFFFFFFFFull) return FS_ERR_SHAPE;  // flat is 32-bit
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (K > c->k_cap) {
    FS_TRY(grow(c, c->states, (size_t)K)); FS_TRY(grow(c, c->ginfo, (size_t)K));
    FS_TRY(grow(c, c->grec, (size_t)K + FS_CHUNK)); FS_TRY(grow(c, c->gsort, (size_t)K + FS_CHUNK));
    FS_TRY(grow(c, c->dsort, (size_t)K + FS_CHUNK)); FS_TRY(grow(c, c->dsuf, (size_t)K / FS_CHUNK + 8 + ((size_t)K + FS_CHUNK) / 2 + 1));
    FS_TRY(grow(c, c->ctr, ((size_t)K / FS_CHUNK + 2) * ((FS_MAX_F + 63) / 64)));   // one counter per (slice, column block)
    FS_TRY(grow(c, c->warm_item, (size_t)K * FS_RMAX));
    c->k_cap = K; c->consol_cap = 0;
  }
  const size_t na = (size_t)K * FS_NVAR * c->d.F;
  if (na > c->gA_cap) { FS_TRY(grow(c, c->gA, na)); c->gA_cap = na; }
  c->Kpad = (K + FS_CHUNK - 1) / FS_CHUNK * FS_CHUNK; c->FT = c->d.F <= 64 ? (c->d.F + 31) / 32 * 32 : (c->d.F + 63) / 64 * 64;   // gA0 row stride: whole column blocks
  const size_t na0 = (size_t)c->Kpad * c->FT;
  if (na0 > c->gA0_cap) { FS_TRY(grow(c, c->gA0, na0)); c->gA0_cap = na0; }
  if (c->d.M > c->warm_m_cap) {
    FS_TRY(grow(c, c->warm_off, (size_t)c->d.M + 1)); FS_TRY(grow(c, c->warm_cursor, (size_t)c->d.M));
    c->warm_m_cap = c->d.M;
  }
  c->K = K; c->have_state = false; c->place_ready = false;
  if (K > 0) {
    FS_CUDA(c, cudaMemcpyAsync(c->states, states, (size_t)K * sizeof(fs_gpu_state), in_kind(space), st));
    FsView v = view_of(c);
    c->launches += fsk_summary(v, c->ginfo, c->gA, c->grec, c->gA0,
                               reinterpret_cast<float*>(c->dsuf + c->Kpad / FS_CHUNK + 4), st, c->timing ? &c->tm : nullptr);
    FS_TRY(check_kernel(c));
  }
  c->have_state = true;
  return pending;
}

int fs_place_batch(fs_ctx* c, int32_t R, const fs_request* reqs, fs_placement* out, int space,
                   void* cuda_stream) {
  if (!c || R < 0 || (R > 0 && (!reqs || !out))) return FS_ERR_ARG;
  if (!space_ok(space)) return FS_ERR_ARG;
  if (!c->have_prof || !c->have_state) return FS_ERR_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (R == 0) return pending;
  if (R > c->r_cap) {
    FS_TRY(grow(c, c->keys, (size_t)R)); FS_TRY(grow(c, c->reqs_dev, (size_t)R));
    FS_TRY(grow(c, c->place_dev, (size_t)R));
    c->r_cap = R;
  }
  const fs_request* d_reqs = reqs; fs_placement* d_out = out;
  // page-locked buffers are mapped into the device's address space: the scoring kernel reads each request
  // and writes each record over PCIe itself (at pod 65,536 x 32 B each way hide behind the scoring; a bulk copy
  // before and after the kernel would sit on the step's critical path)
  bool zero_copy = false;
  if (space == FS_HOST_PINNED && c->zero_copy) {
    cudaPointerAttributes a_in{}, a_out{};
    if (cudaPointerGetAttributes(&a_in, reqs) == cudaSuccess && cudaPointerGetAttributes(&a_out, out) == cudaSuccess &&
        a_in.type == cudaMemoryTypeHost && a_out.type == cudaMemoryTypeHost && a_in.devicePointer && a_out.devicePointer) {
      d_reqs = static_cast<const fs_request*>(a_in.devicePointer);
      d_out = static_cast<fs_placement*>(a_out.devicePointer);
      zero_copy = true;
    } else {
      (void)cudaGetLastError();
    }
  }
  if (space != FS_DEVICE && !zero_copy) {
    FS_CUDA(c, cudaMemcpyAsync(c->reqs_dev, reqs, (size_t)R * sizeof(fs_request), cudaMemcpyHostToDevice, st));
    d_reqs = c->reqs_dev; d_out = c->place_dev;
  }
  FS_TRY(place_prepare(c, st));
  FsPlaceScratch sc{c->keys, c->stats, c->ctr, c->warm_off, c->warm_item, c->sm_count, c->count_work};
  c->launches += fsk_place(view_of(c), R, d_reqs, d_out, sc, st, c->timing ? &c->tm : nullptr);
  FS_TRY(check_kernel(c));
  if (zero_copy) return pending;
  if (space != FS_DEVICE) {
    FS_CUDA(c, cudaMemcpyAsync(out, c->place_dev, (size_t)R * sizeof(fs_placement), cudaMemcpyDeviceToHost, st));
    if (space == FS_HOST_PINNED) return pending;   // the caller synchronises; flags surface on the next call
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_local_config(fs_ctx* c, int32_t n, const int32_t* gpu_ids, uint32_t flags, fs_local_cfg* out,
                    int space, void* cuda_stream) {
  if (!c || n < 0 || (n > 0 && !out) || (flags & ~3u)) return FS_ERR_ARG;
  if (!space_ok(space)) return FS_ERR_ARG;
  if (!c->have_prof || !c->have_state) return FS_ERR_STATE;
  if (!gpu_ids && n > c->K) return FS_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (n == 0) return pending;
  const size_t rows = (size_t)c->d.F * c->d.S;
  const size_t need = (size_t)n * FS_RMAX * 2 * rows;
  if (need > c->local_cap) { FS_TRY(grow(c, c->G, need)); c->local_cap = need; }
  if (n > c->n_cap) {
    FS_TRY(grow(c, c->ids_dev, (size_t)n)); FS_TRY(grow(c, c->local_dev, (size_t)n));
    FS_TRY(grow(c, c->lslots, (size_t)n * FS_RMAX * 2));
    c->n_cap = n;
  }
  if (c->d.M > c->bin_m_cap) {
    FS_TRY(grow(c, c->bin_off, (size_t)c->d.M * 2 * FS_LOCAL_QB + 1)); FS_TRY(grow(c, c->bin_cursor, (size_t)c->d.M * 2 * FS_LOCAL_QB));
    FS_TRY(grow(c, c->keylist, (size_t)c->d.M * 2)); FS_TRY(grow(c, c->nkeys, (size_t)1));
    c->bin_m_cap = c->d.M;
  }
  const int32_t* d_ids = gpu_ids; fs_local_cfg* d_out = out;
  if (space != FS_DEVICE) {
    if (gpu_ids) {
      FS_CUDA(c, cudaMemcpyAsync(c->ids_dev, gpu_ids, (size_t)n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
      d_ids = c->ids_dev;
    }
    d_out = c->local_dev;
  }
  FsLocalScratch sc{c->G, c->comp, c->comp_n, c->ns_stride, c->bin_off, c->bin_cursor, c->keylist, c->nkeys, c->lslots};
  c->launches += fsk_local(view_of(c), n, d_ids, flags, d_out, sc, st, c->timing ? &c->tm : nullptr);
  FS_TRY(check_kernel(c));
  if (space != FS_DEVICE) {
    FS_CUDA(c, cudaMemcpyAsync(out, c->local_dev, (size_t)n * sizeof(fs_local_cfg), cudaMemcpyDeviceToHost, st));
    if (space == FS_HOST_PINNED) return pending;   // the caller synchronises; flags surface on the next call
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_consolidate(fs_ctx* c, fs_consol_out* out, int space, void* cuda_stream) {
  if (!c || !space_ok(space)) return FS_ERR_ARG;
  if (!c->have_prof || !c->have_state) return FS_ERR_STATE;
  if (c->K > 0 && !out) return FS_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (c->K == 0) return pending;
  const size_t kf = (size_t)c->K * c->d.F;
  if (kf > c->consol_cap) {
    const size_t kp = (size_t)c->K * ((c->d.F + 1) / 2 + 1);   // frequency pairs + one row: the pair kernel prefetches one trip ahead
    FS_TRY(grow(c, c->need, kf)); FS_TRY(grow(c, c->E, kf)); FS_TRY(grow(c, c->agg, (size_t)c->K));
    FS_TRY(grow(c, c->E2, kp)); FS_TRY(grow(c, c->T2, kp));
    // the pair kernel's software pipeline loads one row past the last frequency pair and discards it: that row
    // is never written by the pack kernel, so give it defined contents once (no uninitialised read)
    FS_CUDA(c, cudaMemsetAsync(c->E2, 0, kp * sizeof(*c->E2), st)); FS_CUDA(c, cudaMemsetAsync(c->T2, 0, kp * sizeof(*c->T2), st));
    FS_TRY(grow(c, c->ckeys, (size_t)c->K)); FS_TRY(grow(c, c->consol_dev, (size_t)c->K));
    c->consol_cap = kf;
  }
  fs_consol_out* d_out = space != FS_DEVICE ? c->consol_dev : out;
  FsConsolScratch sc{c->need, c->E, c->E2, c->T2, c->agg, c->ckeys};
  c->launches += fsk_consolidate(view_of(c), c->prm, d_out, sc, st, c->timing ? &c->tm : nullptr);
  FS_TRY(check_kernel(c));
  if (space != FS_DEVICE) {
    FS_CUDA(c, cudaMemcpyAsync(out, c->consol_dev, (size_t)c->K * sizeof(fs_consol_out), cudaMemcpyDeviceToHost, st));
    if (space == FS_HOST_PINNED) return pending;   // the caller synchronises; flags surface on the next call
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_dispatch(fs_ctx* c, int32_t R, const fs_request* reqs, fs_placement* out, int space,
                void* cuda_stream) {
  if (!c || R < 0 || (R > 0 && (!reqs || !out))) return FS_ERR_ARG;
  if (!space_ok(space)) return FS_ERR_ARG;
  if (!c->have_prof || !c->have_state) return FS_ERR_STATE;
  if (c->K >= (1 << 24)) return FS_ERR_SHAPE;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (R == 0) return pending;
  if (R > c->r_cap) {
    FS_TRY(grow(c, c->keys, (size_t)R)); FS_TRY(grow(c, c->reqs_dev, (size_t)R));
    FS_TRY(grow(c, c->place_dev, (size_t)R));
    c->r_cap = R;
  }
  const fs_request* d_reqs = reqs; fs_placement* d_out = out;
  if (space != FS_DEVICE) {
    FS_CUDA(c, cudaMemcpyAsync(c->reqs_dev, reqs, (size_t)R * sizeof(fs_request), cudaMemcpyHostToDevice, st));
    d_reqs = c->reqs_dev; d_out = c->place_dev;
  }
  FS_TRY(place_prepare(c, st));
  c->launches += fsk_dispatch(view_of(c), R, d_reqs, d_out, c->warm_off, c->warm_item, st, c->timing ? &c->tm : nullptr);
  FS_TRY(check_kernel(c));
  if (space != FS_DEVICE) {
    FS_CUDA(c, cudaMemcpyAsync(out, c->place_dev, (size_t)R * sizeof(fs_placement), cudaMemcpyDeviceToHost, st));
    if (space == FS_HOST_PINNED) return pending;   // the caller synchronises; flags surface on the next call
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

static int a1_reserve(fs_ctx* c, size_t bytes) {
  if (bytes > c->a1_cap) { FS_TRY(grow(c, c->a1_buf, bytes)); c->a1_cap = bytes; }
  return FS_OK;
}

int fs_dispatch_commit(fs_ctx* c, int32_t R, const fs_request* reqs, fs_placement* out, fs_gpu_avail* after,
                       int space, void* cuda_stream) {
  if (!c || R < 0 || (R > 0 && (!reqs || !out))) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  if (!c->have_prof || !c->have_state) return FS_ERR_STATE;
  if (c->K >= (1 << 24)) return FS_ERR_SHAPE;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (R == 0 && !after) return pending;
  if (R > c->r_cap) {
    FS_TRY(grow(c, c->keys, (size_t)R)); FS_TRY(grow(c, c->reqs_dev, (size_t)R));
    FS_TRY(grow(c, c->place_dev, (size_t)R));
    c->r_cap = R;
  }
  const fs_request* d_reqs = reqs; fs_placement* d_out = out; fs_gpu_avail* d_work = after;
  const size_t wb = (size_t)(c->K > 0 ? c->K : 1) * sizeof(fs_gpu_avail);
  if (space == FS_HOST || !after) {
    FS_TRY(a1_reserve(c, wb));
    d_work = reinterpret_cast<fs_gpu_avail*>(c->a1_buf);
  }
  if (space == FS_HOST && R > 0) {
    FS_CUDA(c, cudaMemcpyAsync(c->reqs_dev, reqs, (size_t)R * sizeof(fs_request), cudaMemcpyHostToDevice, st));
    d_reqs = c->reqs_dev; d_out = c->place_dev;
  }
  c->launches += fsk_dispatch_commit(view_of(c), R, d_reqs, d_out, d_work, st, c->timing ? &c->tm : nullptr);
  FS_TRY(check_kernel(c));
  if (space == FS_HOST) {
    if (R > 0) FS_CUDA(c, cudaMemcpyAsync(out, c->place_dev, (size_t)R * sizeof(fs_placement), cudaMemcpyDeviceToHost, st));
    if (after && c->K > 0) FS_CUDA(c, cudaMemcpyAsync(after, d_work, (size_t)c->K * sizeof(fs_gpu_avail), cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_llm_profiles(fs_ctx* c, int32_t n, const fs_llm* llms, fs_llm_profile* out, int space, void* cuda_stream) {
  if (!c || n < 0 || (n > 0 && (!llms || !out))) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  if (!c->have_prof) return FS_ERR_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (n == 0) return pending;
  const fs_llm* d_in = llms; fs_llm_profile* d_out = out;
  if (space == FS_HOST) {
    FS_TRY(a1_reserve(c, (size_t)n * (sizeof(fs_llm) + sizeof(fs_llm_profile))));
    d_in = reinterpret_cast<fs_llm*>(c->a1_buf);
    d_out = reinterpret_cast<fs_llm_profile*>(c->a1_buf + (size_t)n * sizeof(fs_llm));
    FS_CUDA(c, cudaMemcpyAsync(c->a1_buf, llms, (size_t)n * sizeof(fs_llm), cudaMemcpyHostToDevice, st));
  }
  c->launches += fsk_llm_profile(view_of(c), n, d_in, d_out, st);
  FS_TRY(check_kernel(c));
  if (space == FS_HOST) {
    FS_CUDA(c, cudaMemcpyAsync(out, d_out, (size_t)n * sizeof(fs_llm_profile), cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_ewr(fs_ctx* c, int32_t n, const int32_t* gpu_of, const float* f_mhz, const float* t_ms, int32_t K,
           float* f_gpu, double* out3, int space, void* cuda_stream) {
  if (!c || n < 0 || K < 0 || !out3 || (n > 0 && (!gpu_of || !f_mhz || !t_ms)) || (K > 0 && !f_gpu)) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  const int32_t* d_g = gpu_of; const float *d_f = f_mhz, *d_t = t_ms; float* d_fg = f_gpu; double* d_o = out3;
  if (space == FS_HOST) {
    const size_t nn = (size_t)n, kk = (size_t)K;
    FS_TRY(a1_reserve(c, 32 + nn * 12 + kk * 4 + 16));
    d_o = reinterpret_cast<double*>(c->a1_buf);                       // 3 doubles (32 bytes reserved)
    d_g = reinterpret_cast<int32_t*>(c->a1_buf + 32);
    d_f = reinterpret_cast<float*>(c->a1_buf + 32 + nn * 4);
    d_t = reinterpret_cast<float*>(c->a1_buf + 32 + nn * 8);
    d_fg = reinterpret_cast<float*>(c->a1_buf + 32 + nn * 12);
    if (n > 0) {
      FS_CUDA(c, cudaMemcpyAsync((void*)d_g, gpu_of, nn * 4, cudaMemcpyHostToDevice, st));
      FS_CUDA(c, cudaMemcpyAsync((void*)d_f, f_mhz, nn * 4, cudaMemcpyHostToDevice, st));
      FS_CUDA(c, cudaMemcpyAsync((void*)d_t, t_ms, nn * 4, cudaMemcpyHostToDevice, st));
    }
  }
  c->launches += fsk_ewr(n, d_g, d_f, d_t, K, d_fg, d_o, c->flag_dev, st);
  FS_TRY(check_kernel(c));
  if (space == FS_HOST) {
    if (K > 0) FS_CUDA(c, cudaMemcpyAsync(f_gpu, d_fg, (size_t)K * 4, cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaMemcpyAsync(out3, d_o, 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_replace_plan(fs_ctx* c, int32_t n, const fs_plan_llm* llms, int32_t s_eff, float m_eff,
                    int32_t* gpu_of, int32_t* summary, int space, void* cuda_stream) {
  if (!c || n < 0 || !summary || (n > 0 && (!llms || !gpu_of)) || s_eff < 1 || s_eff > FS_MAX_S) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  const size_t sb = fsk_plan_scratch_bytes(n);
  if (sb > c->pl_cap) { FS_TRY(grow(c, c->pl_buf, sb)); c->pl_cap = sb; }
  const fs_plan_llm* d_in = llms; int32_t* d_g = gpu_of; int32_t* d_s = summary;
  if (space == FS_HOST) {
    const size_t nn = (size_t)n;
    FS_TRY(a1_reserve(c, 16 + nn * (sizeof(fs_plan_llm) + 4)));
    d_s = reinterpret_cast<int32_t*>(c->a1_buf);
    d_in = reinterpret_cast<fs_plan_llm*>(c->a1_buf + 16);
    d_g = reinterpret_cast<int32_t*>(c->a1_buf + 16 + nn * sizeof(fs_plan_llm));
    if (n > 0) FS_CUDA(c, cudaMemcpyAsync((void*)d_in, llms, nn * sizeof(fs_plan_llm), cudaMemcpyHostToDevice, st));
  }
  c->launches += fsk_replace_plan(n, d_in, s_eff, m_eff, c->pl_buf, d_g, d_s, c->flag_dev, st);
  FS_TRY(check_kernel(c));
  if (space == FS_HOST) {
    if (n > 0) FS_CUDA(c, cudaMemcpyAsync(gpu_of, d_g, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaMemcpyAsync(summary, d_s, 16, cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_migration_plan(fs_ctx* c, int32_t n, const float* bytes_mb, const float* bw, int32_t* dst_of,
                      int64_t* total_us, int space, void* cuda_stream) {
  if (!c || n < 0 || !total_us || (n > 0 && (!bytes_mb || !bw || !dst_of))) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  if (n > 1024) return FS_ERR_SHAPE;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  const float *d_b = bytes_mb, *d_w = bw; int32_t* d_d = dst_of; long long* d_t = reinterpret_cast<long long*>(total_us);
  if (space == FS_HOST) {
    const size_t nn = (size_t)n;
    FS_TRY(a1_reserve(c, 16 + nn * 8 + nn * nn * 4));
    d_t = reinterpret_cast<long long*>(c->a1_buf);
    d_b = reinterpret_cast<float*>(c->a1_buf + 16); d_d = reinterpret_cast<int32_t*>(c->a1_buf + 16 + nn * 4);
    d_w = reinterpret_cast<float*>(c->a1_buf + 16 + nn * 8);
    if (n > 0) {
      FS_CUDA(c, cudaMemcpyAsync((void*)d_b, bytes_mb, nn * 4, cudaMemcpyHostToDevice, st));
      FS_CUDA(c, cudaMemcpyAsync((void*)d_w, bw, nn * nn * 4, cudaMemcpyHostToDevice, st));
    }
  }
  c->launches += fsk_assign(n, d_b, d_w, d_d, d_t, c->flag_dev, st);
  FS_TRY(check_kernel(c));
  if (space == FS_HOST) {
    if (n > 0) FS_CUDA(c, cudaMemcpyAsync(dst_of, d_d, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaMemcpyAsync(total_us, d_t, 8, cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_migration_select(fs_ctx* c, int32_t r, const fs_mig_req* reqs, uint8_t* flags, float* mig_ms, int space,
                        void* cuda_stream) {
  if (!c || r < 0 || (r > 0 && (!reqs || !flags || !mig_ms))) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (r == 0) return pending;
  const fs_mig_req* d_q = reqs; uint8_t* d_f = flags; float* d_m = mig_ms;
  if (space == FS_HOST) {
    const size_t rr = (size_t)r;
    FS_TRY(a1_reserve(c, rr * (sizeof(fs_mig_req) + 4 + 1) + 16));
    d_q = reinterpret_cast<fs_mig_req*>(c->a1_buf); d_m = reinterpret_cast<float*>(c->a1_buf + rr * sizeof(fs_mig_req));
    d_f = c->a1_buf + rr * (sizeof(fs_mig_req) + 4);
    FS_CUDA(c, cudaMemcpyAsync((void*)d_q, reqs, rr * sizeof(fs_mig_req), cudaMemcpyHostToDevice, st));
  }
  c->launches += fsk_migration_select(r, d_q, d_f, d_m, st);
  FS_TRY(check_kernel(c));
  if (space == FS_HOST) {
    FS_CUDA(c, cudaMemcpyAsync(flags, d_f, (size_t)r, cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaMemcpyAsync(mig_ms, d_m, (size_t)r * 4, cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

int fs_batch_tasks(fs_ctx* c, int32_t n, const int32_t* gpu_ids, const int32_t* task_off,
                   const fs_task* tasks, fs_task_out* out, int32_t n_tasks, int space, void* cuda_stream) {
  if (!c || n < 0 || n_tasks < 0 || (n > 0 && !task_off) || (n_tasks > 0 && (!tasks || !out))) return FS_ERR_ARG;
  if (space != FS_HOST && space != FS_DEVICE) return FS_ERR_ARG;
  if (!c->have_prof || !c->have_state) return FS_ERR_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream; c->cur = st;
  FS_CUDA(c, cudaSetDevice(c->dev));
  const int pending = take_flags(c);
  if (n == 0) return pending;
  const int32_t* d_ids = gpu_ids; const int32_t* d_off = task_off; const fs_task* d_tasks = tasks; fs_task_out* d_out = out;
  if (space == FS_HOST) {
    if (task_off[0] != 0 || task_off[n] != n_tasks) return FS_ERR_ARG;
    if (n > c->bt_n_cap) { FS_TRY(grow(c, c->bt_ids, (size_t)n)); FS_TRY(grow(c, c->bt_off, (size_t)n + 1)); c->bt_n_cap = n; }
    if (n_tasks > c->bt_t_cap) { FS_TRY(grow(c, c->bt_tasks, (size_t)n_tasks)); FS_TRY(grow(c, c->bt_out, (size_t)n_tasks)); c->bt_t_cap = n_tasks; }
    if (gpu_ids) { FS_CUDA(c, cudaMemcpyAsync(c->bt_ids, gpu_ids, (size_t)n * sizeof(int32_t), cudaMemcpyHostToDevice, st)); d_ids = c->bt_ids; }
    FS_CUDA(c, cudaMemcpyAsync(c->bt_off, task_off, ((size_t)n + 1) * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (n_tasks > 0) FS_CUDA(c, cudaMemcpyAsync(c->bt_tasks, tasks, (size_t)n_tasks * sizeof(fs_task), cudaMemcpyHostToDevice, st));
    d_off = c->bt_off; d_tasks = c->bt_tasks; d_out = c->bt_out;
  }
  c->launches += fsk_batch_tasks(view_of(c), n, d_ids, d_off, d_tasks, d_out, n_tasks, st, c->timing ? &c->tm : nullptr);
  FS_TRY(check_kernel(c));
  if (space == FS_HOST) {
    if (n_tasks > 0) FS_CUDA(c, cudaMemcpyAsync(out, c->bt_out, (size_t)n_tasks * sizeof(fs_task_out), cudaMemcpyDeviceToHost, st));
    FS_CUDA(c, cudaStreamSynchronize(st));
    const int now = take_flags(c);
    return pending != FS_OK ? pending : now;
  }
  return pending;
}

const char* fs_strerror(int code) {
  switch (code) {
    case FS_OK: return "ok";
    case FS_ERR_ARG: return "bad argument";
    case FS_ERR_SHAPE: return "dims outside the supported range";
    case FS_ERR_STATE: return "profiles or GPU state not loaded (or the call must allocate while its stream is being captured)";
    case FS_ERR_RANGE: return "index or value out of range in device data";
    case FS_ERR_CUDA: return "CUDA runtime error";
    case FS_ERR_NOMEM: return "out of memory";
    default: return "unknown";
  }
}

int fs_last_cuda_error(const fs_ctx* c) { return c ? c->last_cuda : 0; }
uint64_t fs_launch_count(const fs_ctx* c) { return c ? c->launches : 0; }

int fs_set_timing(fs_ctx* c, int on) {
  if (!c) return FS_ERR_ARG;
  FS_CUDA(c, cudaSetDevice(c->dev));
  if (on && !c->have_events) {
    for (int i = 0; i < FS_T_COUNT; ++i) {
      FS_CUDA(c, cudaEventCreate(&c->tm.beg[i])); FS_CUDA(c, cudaEventCreate(&c->tm.end[i]));
      c->tm.used[i] = false;
    }
    c->have_events = true;
  }
  c->timing = on != 0;
  return FS_OK;
}

int fs_get_timing(fs_ctx* c, float* ms, int n) {
  if (!c || !ms || n < 0) return FS_ERR_ARG;
  FS_CUDA(c, cudaSetDevice(c->dev));
  for (int i = 0; i < n; ++i) {
    ms[i] = -1.0f;
    if (i < FS_T_COUNT && c->have_events && c->tm.used[i]) {
      FS_CUDA(c, cudaEventSynchronize(c->tm.end[i]));
      FS_CUDA(c, cudaEventElapsedTime(&ms[i], c->tm.beg[i], c->tm.end[i]));
    }
  }
  return FS_OK;
}

int fs_set_work_stats(fs_ctx* c, int on) {
  if (!c) return FS_ERR_ARG;
  c->count_work = on != 0;
  return FS_OK;
}

int fs_last_place_stats(fs_ctx* c, uint64_t out[FS_NSTATS]) {
  if (!c || !out) return FS_ERR_ARG;
  unsigned long long h[FS_NSTATS] = {};
  FS_CUDA(c, cudaSetDevice(c->dev));
  FS_CUDA(c, cudaMemcpy(h, c->stats, sizeof(h), cudaMemcpyDeviceToHost));
  for (int i = 0; i < FS_NSTATS; ++i) out[i] = h[i];
  return FS_OK;
}

}  // extern "C"
