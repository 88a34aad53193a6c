// fs_plan.cu — fs_replace_plan: Algorithm 1, phases 2-3 (prose P:341-357).
//
// Phase 2: N_sm, N_mem by Best-Fit-Decreasing against (S_eff, M_eff), N_min = max.  Phase 3: LLMs in
// ascending l.F; Target / Candidate = the two GPUs with the closest operating frequency (an empty GPU is
// at distance +INF); direct placement, EWR-driven swap of the target's lowest-frequency resident, the
// candidate, the closest other GPU that fits, a new GPU (DESIGN.md s32 for the readings).
//
// The loop over LLMs is sequential by definition (every step depends on the GPUs the previous ones
// filled); what is parallel is inside a step: the searches over bins / GPUs run lane <-> GPU with
// 64-bit (value, index) keys reduced by shuffles, the three orders are rank sorts (lane <-> item).
// One warp does the whole plan; the per-GPU resident lists hold at most S_eff <= 32 entries, so the
// waste sums of the swap test are short and are taken by lane 0 in the order the definition fixes.
#include <mutex>

#include "fs_kernels.h"

namespace {

constexpr int PL_RES = FS_MAX_S;      // residents per GPU at most (every LLM needs >= 1 share unit)

struct PlanScratch {
  int32_t* order;     // [n]      items in processing order
  int32_t* rem_u;     // [n]      BFD: remaining units per bin
  float* rem_m;       // [n]      BFD: remaining memory per bin
  int32_t* sm_left;   // [2n+1]
  float* mem_left;    // [2n+1]
  float* freq;        // [2n+1]
  int32_t* cnt;       // [2n+1]
  int32_t* res;       // [2n+1][PL_RES]
};

// mode 0 (units BFD): fits a GPU's units; mode 1 (memory BFD): fits its memory; mode 2 (placement): both
__device__ __forceinline__ bool placeable(const fs_plan_llm& l, int s_eff, float m_eff, int mode) {
  const bool u = l.need_units >= 1 && l.need_units <= s_eff, m = l.mem_mb <= m_eff;
  return mode == 0 ? u : mode == 1 ? m : (u && m);
}

// order[] = the placeable items sorted by key (ascending), ties by lower index; returns their count.
// mode 0: decreasing units, 1: decreasing memory, 2: ascending frequency.
__device__ int rank_order(const fs_plan_llm* L, int n, int s_eff, float m_eff, int mode, int32_t* order, int lane) {
  int total = 0;
  for (int base = 0; base < n; base += 32) {
    const int i = base + lane;
    const bool live = i < n && placeable(L[i], s_eff, m_eff, mode);
    total += __popc(__ballot_sync(0xffffffffu, live));
  }
  for (int base = 0; base < n; base += 32) {
    const int i = base + lane;
    const bool live = i < n && placeable(L[i], s_eff, m_eff, mode);
    if (live) {
      const fs_plan_llm me = L[i];
      int rank = 0;
      for (int j = 0; j < n; ++j) {
        const fs_plan_llm o = L[j];
        if (!placeable(o, s_eff, m_eff, mode)) continue;
        bool before;
        if (mode == 0) before = o.need_units > me.need_units || (o.need_units == me.need_units && j < i);
        else if (mode == 1) before = o.mem_mb > me.mem_mb || (o.mem_mb == me.mem_mb && j < i);
        else before = o.f_mhz < me.f_mhz || (o.f_mhz == me.f_mhz && j < i);
        rank += before ? 1 : 0;
      }
      order[rank] = i;
    }
  }
  __syncwarp();
  return total;
}

__device__ __forceinline__ double waste_of(const fs_plan_llm* L, const int32_t* res, int cnt, int skip, int extra) {
  float F = 0.0f;
  for (int x = 0; x < cnt; ++x) if (res[x] != skip && L[res[x]].f_mhz > F) F = L[res[x]].f_mhz;
  if (extra >= 0 && L[extra].f_mhz > F) F = L[extra].f_mhz;
  const double F3 = (double)F * F * F;
  double w = 0.0;
  for (int x = 0; x < cnt; ++x) if (res[x] != skip) { const double f = L[res[x]].f_mhz; w += (double)L[res[x]].t_ms * (F3 - f * f * f); }
  if (extra >= 0) { const double f = L[extra].f_mhz; w += (double)L[extra].t_ms * (F3 - f * f * f); }
  return w;
}

__global__ void __launch_bounds__(32) replace_plan_kernel(int n, const fs_plan_llm* __restrict__ L, int s_eff, float m_eff,
                                                         PlanScratch sc, int32_t* __restrict__ gpu_of,
                                                         int32_t* __restrict__ summary, int* flag) {
  const int lane = threadIdx.x;
  bool bad = false;
  for (int i = lane; i < n; i += 32) { gpu_of[i] = -1; bad = bad || L[i].need_units < 1; }
  if (__any_sync(0xffffffffu, bad) && lane == 0) fs_raise(flag, FS_FLAG_ARG);
  // ---- phase 2: Best-Fit-Decreasing on units, then on memory ------------------------------------
  int nbins[2];
  for (int mode = 0; mode < 2; ++mode) {
    const int m = rank_order(L, n, s_eff, m_eff, mode, sc.order, lane);
    int bins = 0;
    for (int a = 0; a < m; ++a) {
      const fs_plan_llm it = L[sc.order[a]];
      unsigned long long key = FS_KEY_NONE;            // (remaining room, bin): the fullest bin that fits
      for (int g = lane; g < bins; g += 32) {
        if (mode == 0) { const int r = sc.rem_u[g]; if (r >= it.need_units) { const unsigned long long k = ((unsigned long long)(uint32_t)r << 32) | (uint32_t)g; key = k < key ? k : key; } }
        else { const float r = sc.rem_m[g]; if (r >= it.mem_mb) { const unsigned long long k = fs_make_key(r, (uint32_t)g); key = k < key ? k : key; } }
      }
      key = fs_warp_min_key(key);
      if (lane == 0) {
        int g = (int)(uint32_t)key;
        if (key == FS_KEY_NONE) { g = bins; sc.rem_u[g] = s_eff; sc.rem_m[g] = m_eff; }
        if (mode == 0) sc.rem_u[g] -= it.need_units; else sc.rem_m[g] = __fsub_rn(sc.rem_m[g], it.mem_mb);
      }
      if (key == FS_KEY_NONE) bins += 1;
      __syncwarp();
    }
    nbins[mode] = bins;
  }
  const int n_min = max(nbins[0], nbins[1]);
  // ---- phase 3 -------------------------------------------------------------------------------------
  int G = n_min;
  for (int g = lane; g < 2 * n + 1; g += 32) { sc.sm_left[g] = s_eff; sc.mem_left[g] = m_eff; sc.freq[g] = 0.0f; sc.cnt[g] = 0; }
  const int m = rank_order(L, n, s_eff, m_eff, 2, sc.order, lane);
  for (int a = 0; a < m; ++a) {
    const int l = sc.order[a];
    const fs_plan_llm it = L[l];
    // Target, Candidate: (distance, GPU) keys; lanes also remember the closest GPU that FITS (fallback)
    unsigned long long k1 = FS_KEY_NONE, k2 = FS_KEY_NONE;
    for (int g = lane; g < G; g += 32) {
      const float dist = sc.cnt[g] == 0 ? FS_INF : fabsf(__fsub_rn(sc.freq[g], it.f_mhz));
      const unsigned long long k = fs_make_key(dist, (uint32_t)g);
      if (k < k1) { k2 = k1; k1 = k; } else if (k < k2) k2 = k;
    }
    // warp: smallest and second smallest of the union of the lanes' (k1, k2)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long a1 = __shfl_xor_sync(0xffffffffu, k1, o), a2 = __shfl_xor_sync(0xffffffffu, k2, o);
      const unsigned long long lo = a1 < k1 ? a1 : k1, hi = a1 < k1 ? k1 : a1;   // hi = larger of the two minima
      const unsigned long long s2 = a2 < k2 ? a2 : k2;
      k1 = lo; k2 = hi < s2 ? hi : s2;
    }
    const int tgt = k1 == FS_KEY_NONE ? -1 : (int)(uint32_t)k1, cand = k2 == FS_KEY_NONE ? -1 : (int)(uint32_t)k2;
    int dest = -1, moved = -1;                         // decided by lane 0, then broadcast
    if (lane == 0) {
      auto fits = [&](int g, int who, int fu, float fm, bool freed) {
        const int sm = sc.sm_left[g] + fu;
        const float mem = freed ? __fadd_rn(sc.mem_left[g], fm) : sc.mem_left[g];
        return L[who].need_units <= sm && L[who].mem_mb <= mem;
      };
      if (tgt >= 0 && fits(tgt, l, 0, 0.0f, false)) dest = tgt;
      if (dest < 0 && tgt >= 0 && cand >= 0 && sc.cnt[tgt] > 0) {
        const int32_t* rt = sc.res + (size_t)tgt * PL_RES;
        int lo = -1;
        for (int x = 0; x < sc.cnt[tgt]; ++x) {
          const int r = rt[x];
          if (lo < 0 || L[r].f_mhz < L[lo].f_mhz || (L[r].f_mhz == L[lo].f_mhz && r < lo)) lo = r;
        }
        const int32_t* rc = sc.res + (size_t)cand * PL_RES;
        const double e_curr = waste_of(L, rt, sc.cnt[tgt], -1, l) + waste_of(L, rc, sc.cnt[cand], -1, -1);
        const double e_swap = waste_of(L, rt, sc.cnt[tgt], lo, l) + waste_of(L, rc, sc.cnt[cand], -1, lo);
        if (fits(cand, lo, 0, 0.0f, false) && fits(tgt, l, L[lo].need_units, L[lo].mem_mb, true) && e_swap < e_curr) {
          dest = tgt; moved = lo;
        }
      }
      if (dest < 0 && cand >= 0 && fits(cand, l, 0, 0.0f, false)) dest = cand;
    }
    dest = __shfl_sync(0xffffffffu, dest, 0); moved = __shfl_sync(0xffffffffu, moved, 0);
    if (dest < 0) {                                    // fallback: the closest other GPU that fits
      unsigned long long kf = FS_KEY_NONE;
      for (int g = lane; g < G; g += 32) {
        if (g == tgt || g == cand) continue;
        if (it.need_units <= sc.sm_left[g] && it.mem_mb <= sc.mem_left[g]) {
          const float dist = sc.cnt[g] == 0 ? FS_INF : fabsf(__fsub_rn(sc.freq[g], it.f_mhz));
          const unsigned long long k = fs_make_key(dist, (uint32_t)g);
          kf = k < kf ? k : kf;
        }
      }
      kf = fs_warp_min_key(kf);
      if (kf != FS_KEY_NONE) dest = (int)(uint32_t)kf;
      else { dest = G; G += 1; }                       // activate a new GPU
    }
    if (lane == 0) {
      auto put = [&](int g, int who) {
        sc.sm_left[g] -= L[who].need_units; sc.mem_left[g] = __fsub_rn(sc.mem_left[g], L[who].mem_mb);
        sc.res[(size_t)g * PL_RES + sc.cnt[g]] = who; sc.cnt[g] += 1;
        if (L[who].f_mhz > sc.freq[g]) sc.freq[g] = L[who].f_mhz;
        gpu_of[who] = g;
      };
      if (moved >= 0) {                                // the outlier leaves the target for the candidate
        int32_t* rt = sc.res + (size_t)dest * PL_RES;
        sc.sm_left[dest] += L[moved].need_units; sc.mem_left[dest] = __fadd_rn(sc.mem_left[dest], L[moved].mem_mb);
        int c = 0; float f = 0.0f;
        for (int x = 0; x < sc.cnt[dest]; ++x) if (rt[x] != moved) { rt[c++] = rt[x]; if (L[rt[c - 1]].f_mhz > f) f = L[rt[c - 1]].f_mhz; }
        sc.cnt[dest] = c; sc.freq[dest] = f;
        put(cand, moved);
      }
      put(dest, l);
    }
    __syncwarp();
  }
  if (lane == 0) { summary[0] = nbins[0]; summary[1] = nbins[1]; summary[2] = n_min; summary[3] = G; }
}

}  // namespace

size_t fsk_plan_scratch_bytes(int n) {
  const size_t g = 2 * (size_t)n + 1;
  return sizeof(int32_t) * ((size_t)n * 2 + g * 2 + g * PL_RES) + sizeof(float) * ((size_t)n + g * 2) + 256;
}

int fsk_replace_plan(int n, const fs_plan_llm* llms, int s_eff, float m_eff, void* scratch, int32_t* gpu_of,
                     int32_t* summary, int* flag, cudaStream_t st) {
  const size_t g = 2 * (size_t)n + 1;
  unsigned char* p = reinterpret_cast<unsigned char*>(scratch);
  PlanScratch sc;
  auto take = [&](size_t bytes) { void* q = p; p += (bytes + 15) / 16 * 16; return q; };
  sc.order = (int32_t*)take(sizeof(int32_t) * (size_t)max(n, 1)); sc.rem_u = (int32_t*)take(sizeof(int32_t) * (size_t)max(n, 1));
  sc.rem_m = (float*)take(sizeof(float) * (size_t)max(n, 1));
  sc.sm_left = (int32_t*)take(sizeof(int32_t) * g); sc.mem_left = (float*)take(sizeof(float) * g);
  sc.freq = (float*)take(sizeof(float) * g); sc.cnt = (int32_t*)take(sizeof(int32_t) * g);
  sc.res = (int32_t*)take(sizeof(int32_t) * g * PL_RES);
  replace_plan_kernel<<<1, 32, 0, st>>>(n, llms, s_eff, m_eff, sc, gpu_of, summary, flag);
  return 1;
}

// ---- fs_replace_plan_static: the same plan without any allocation -------------------------------------
//
// Who this is for.  fs_replace_plan lives on an fs_ctx, and both fs_create and the first call of a given
// size go through cudaMalloc.  Some hosts of this library cannot do that at the moment they want a plan:
// the scheduler runs inside (or beside) a serving engine that reserved nearly all of HBM for weights and
// KV cache at start-up, so a late cudaMalloc fails or has to be fought for; and a control loop that shares
// the GPU with running inference must not call cudaMalloc / cudaFree at all, because both take the
// driver's allocator lock and cudaFree waits for the whole device, stalling the very streams the scheduler
// is trying not to disturb.  Those callers get this one entry point: it needs no context and never calls
// cudaMalloc, cudaFree, cudaHostAlloc or any routine that allocates.  The caller brings the input and the
// two outputs (device-addressable); the kernel's working arrays (processing order, the BFD bins, the per-GPU
// room / frequency / resident lists) live in the fixed array below.
//
// What it costs.  Every GPU on which this library's code gets loaded holds sizeof(g_plan_static) bytes
// (about 300 KiB, see the static_assert) from module load until the process exits, whether or not the entry
// point is ever called.  The size is fixed at build time, hence the limit n <= FS_PLAN_STATIC_MAX_N.
//
// `g_plan_static` is a DEVICE symbol.  In host code the name is only a handle for the runtime: taking its
// address there yields a host address, and a kernel handed that would fault (or, on a system where the GPU can
// reach host memory, quietly work on the wrong bytes).  The device address comes from cudaGetSymbolAddress,
// asked once per device with that device current (plan_static_base below).
constexpr size_t pl_align16(size_t b) { return (b + 15) / 16 * 16; }
constexpr size_t pl_static_bytes(size_t n) {   // the carve-up of fsk_replace_plan, for n items
  return 3 * pl_align16(4 * n) + 4 * pl_align16(4 * (2 * n + 1)) + pl_align16(4 * (2 * n + 1) * (size_t)FS_MAX_S);
}
constexpr size_t PL_STATIC_HEAD = 256;         // first 256 bytes: the kernel's range-flag words (a sink here)
constexpr size_t PL_STATIC_BYTES = PL_STATIC_HEAD + pl_static_bytes(FS_PLAN_STATIC_MAX_N);
static_assert(PL_STATIC_BYTES <= 320 * 1024, "keep the resident scratch modest");
static __device__ __align__(256) unsigned char g_plan_static[PL_STATIC_BYTES];

namespace {
constexpr int PL_STATIC_MAX_DEV = 64;
std::mutex g_plan_static_mu;
unsigned char* g_plan_static_base[PL_STATIC_MAX_DEV];   // device address of g_plan_static, per device ordinal

// Device address of the scratch array on the CURRENT device (first use on a device: one
// cudaGetSymbolAddress, which also makes the runtime load this library's code onto that device).
int plan_static_base(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return FS_ERR_CUDA; }
  if (dev < 0 || dev >= PL_STATIC_MAX_DEV) return FS_ERR_SHAPE;
  std::lock_guard<std::mutex> lock(g_plan_static_mu);
  if (!g_plan_static_base[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_plan_static) != cudaSuccess || !p) { cudaGetLastError(); return FS_ERR_CUDA; }
    g_plan_static_base[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_plan_static_base[dev];
  return FS_OK;
}
}  // namespace

extern "C" int fs_replace_plan_static(int32_t n, const fs_plan_llm* llms, int32_t s_eff, float m_eff,
                                      int32_t* gpu_of, int32_t* summary, void* cuda_stream) {
  if (n < 0 || !summary || (n > 0 && (!llms || !gpu_of)) || s_eff < 1 || s_eff > FS_MAX_S) return FS_ERR_ARG;
  if (n > FS_PLAN_STATIC_MAX_N) return FS_ERR_SHAPE;     // the resident array is sized for FS_PLAN_STATIC_MAX_N
  unsigned char* base = nullptr;
  const int rc = plan_static_base(&base);
  if (rc != FS_OK) return rc;
  // Nothing in the array has to start at zero: the kernel writes every word before it reads it (order[] by
  // the rank sort, a bin's room when the bin is opened, the per-GPU records up to 2n+1 at the top of phase
  // 3, a resident list only below its count), so whatever the previous call left behind is never seen.
  fsk_replace_plan(n, llms, s_eff, m_eff, base + PL_STATIC_HEAD, gpu_of, summary, reinterpret_cast<int*>(base),
                   static_cast<cudaStream_t>(cuda_stream));
  if (cudaGetLastError() != cudaSuccess) return FS_ERR_CUDA;
  return FS_OK;
}
