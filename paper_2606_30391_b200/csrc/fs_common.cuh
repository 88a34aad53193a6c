// fs_common.cuh — device-side building blocks of libfestina_eval (sm_100a).
//
// The product path.  Shares no code with oracle/ (own structs via include/festina_eval.h, own
// arithmetic).  Every fl(.) of DESIGN.md "Numerics" is ONE binary32 round-to-nearest-even
// operation: products and sums go through __fmul_rn/__fadd_rn/__fsub_rn, which nvcc never
// contracts into FMA.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/festina_eval.h"

#define FS_INF __int_as_float(0x7f800000)
#define FS_NEED_INF 255          // "no feasible share" marker of the consolidation need[] bytes
#define FS_NVAR (FS_RMAX + 1)    // co-resident energy variants: 0 = as is, 1+j = bump tenant j
#define FS_KEY_NONE 0xFFFFFFFFFFFFFFFFull

// Sticky range-error words: int[4] in mapped (zero-copy) host memory, one word per source.
// Kernels only ever store 1 (plain store; no PCIe atomics needed); the next API call reads
// and clears them on the host.
enum { FS_FLAG_TABLE = 0, FS_FLAG_STATE = 1, FS_FLAG_REQUEST = 2, FS_FLAG_ARG = 3, FS_NFLAGS = 4 };
__device__ __forceinline__ void fs_raise(int* flag, int which) {
  *((volatile int*)flag + which) = 1;
}

// Per-GPU summary written by the summary kernel (fs_set_gpu_state) and read by placement.
// 48 bytes, 16-byte aligned so that one GPU is three 128-bit loads.
struct __align__(16) FsGpuInfo {
  float t_avail_ms;     // T_avail
  float mem_free_mb;    // free memory
  float e_cur;          // Ecur: slot-order energy sum at F_curr, no bump (R:s4)
  int32_t n_res;        // 0 = inactive or invalid record
  int32_t sm_free;      // S - sum(sigma_i+1)
  int32_t f_floor;      // lowest phi at which every co-resident is feasible (-1: none)
  int16_t model[FS_RMAX];   // tenant models (-1 beyond n_res)
  int16_t br1[FS_RMAX];     // decode bucket a joining request sees: beta_1+1 if q_1>0 else 0;
                            // -1 = bucket past the table (candidate dropped)
  int32_t f_cur;            // F_curr (0 for an inactive / invalid record)
  uint32_t _pad;
};
static_assert(sizeof(FsGpuInfo) == 48, "FsGpuInfo layout");

// Compact per-GPU record the dense placement kernel stages with TMA (32 bytes).
struct __align__(16) FsGpuRec {
  float t_avail_ms, mem_free_mb, e_cur;
  uint32_t meta;            // n_res | sm_free << 8 | F_curr << 16   (n_res == 0: never a candidate)
  int16_t model[FS_RMAX];
  float a_min;              // min over phi of A0[k][phi] (+INF: co-residents never feasible)
  uint32_t k;               // GPU index (the sorted copy is not in index order)
};
static_assert(sizeof(FsGpuRec) == 32, "FsGpuRec layout");
// Prefix minima of one plane (model, phase, batch bucket) over shares <= s and all phi (fs_tables.cu)
struct __align__(16) FsPlaneMin {
  float lpf;                // min of the exact product LAT*POW, times (1 - 2^-22), rounded DOWN to binary32
  float lmin;               // min LAT
  float eta;                // 2^-149 * (max POW + 1), rounded UP
  float _pad;
};
static_assert(sizeof(FsPlaneMin) == 16, "FsPlaneMin layout");
// One (GPU k, tenant slot j) that hosts a model: what a request of that model needs to bound and
// to score the WARM pair (r, k) (64 bytes; built by fs_set_gpu_state, listed per model).
struct __align__(16) FsWarmItem {
  int32_t k, j;
  int32_t br1;              // decode bucket the request joins (-1: past the table)
  int32_t sm_free;
  float t_avail_ms, mem_free_mb, e_cur;
  float a_min;              // min over phi of A[k][1+j][phi]
  float lp1f, eta1, l1_min; // FsPlaneMin of plane (model, decode, br1) at share sm_free - 1
  uint32_t _pad0;
  int32_t f_cur;            // F_curr of the GPU
  uint32_t magic;           // ceil(2^32 / (br1+1)) for br1 >= 1 (0: br1 == 0): rounds by multiply-high
  uint32_t _pad[2];
};
static_assert(sizeof(FsWarmItem) == 64, "FsWarmItem layout");
#define FS_CHUNK 32         // GPUs per staged chunk (one per lane in the eligibility pass)

struct FsDimsDev { int M, F, S, B; };

// ---- table addressing --------------------------------------------------------------------
// logical layout  [M][2][F][S][B]  (beta fastest): the batch search of fs_local_config
__device__ __forceinline__ size_t fs_idx(const FsDimsDev& d, int m, int p, int f, int s, int b) {
  return ((((size_t)m * 2 + p) * d.F + f) * d.S + s) * d.B + b;
}
// plane layout    [M][2][B][S][F]  (phi fastest): one (sigma,phi) plane per (model,phase,beta)
// (the plane's index fits 32 bits: M <= 32767, B <= 256; one widening multiply by S*F <= 8192 forms the offset)
__device__ __forceinline__ size_t fs_plane(const FsDimsDev& d, int m, int p, int b) {
  return (size_t)(uint32_t)((m * 2 + p) * d.B + b) * (size_t)(uint32_t)(d.S * d.F);
}

// ---- arithmetic ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t fs_ceil_div(uint32_t q, uint32_t n) { return (q + n - 1u) / n; }

// 64-bit argmin key: high word = order-preserving transform of the fp32 value, low word = flat
// index (BASELINE north_star; SURVEY §8(c) "Numerics").  -0 is canonicalised to +0 first.
__device__ __forceinline__ uint32_t fs_orderable(float v) {
  if (v == 0.0f) v = 0.0f;
  uint32_t u = __float_as_uint(v);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float fs_unorderable(uint32_t o) {
  uint32_t u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
  return __uint_as_float(u);
}
__device__ __forceinline__ unsigned long long fs_make_key(float v, uint32_t flat) {
  return ((unsigned long long)fs_orderable(v) << 32) | flat;
}
// warp-wide minimum of a 64-bit key by two 32-bit reductions (redux.sync): the high words first, then the low
// words of the lanes that hold the minimal high word (all 32 lanes must call it)
__device__ __forceinline__ uint32_t fs_redux_min_u32(uint32_t x) {
  uint32_t r;
  asm volatile("redux.sync.min.u32 %0, %1, 0xffffffff;" : "=r"(r) : "r"(x));
  return r;
}
__device__ __forceinline__ unsigned long long fs_warp_min_key(unsigned long long k) {
  const uint32_t hi = (uint32_t)(k >> 32), lo = (uint32_t)k;
  const uint32_t mh = fs_redux_min_u32(hi);
  const uint32_t ml = fs_redux_min_u32(hi == mh ? lo : 0xFFFFFFFFu);
  return ((unsigned long long)mh << 32) | ml;
}

// ceil(q / n) for q <= 2^24, 1 <= n <= 256 by multiply-high: magic = ceil(2^32 / n) for n >= 2 (0 stands for
// n == 1).  floor((q-1)/n) = umulhi(q-1, magic) exactly, because (q-1) * (magic*n - 2^32) < 2^24 * 2^8 = 2^32.
// Beyond that it can be one too large (n = 255: first at q = 16,909,560), so a caller whose q may exceed 2^24
// (the padded output length O of a request) tests the range and divides otherwise; tests/test_magic_division.py
// checks the bound and the first failures.
__host__ __device__ __forceinline__ uint32_t fs_magic(uint32_t n) {
  return n <= 1u ? 0u : (uint32_t)((0x100000000ull + n - 1u) / n);
}
__device__ __forceinline__ uint32_t fs_ceil_div_magic(uint32_t q, uint32_t magic) {
  return (magic == 0u || q == 0u) ? q : __umulhi(q - 1u, magic) + 1u;
}

// A lower bound on e = fl(fl(fr*LAT)*POW) of EVERY entry of a plane prefix, fr >= 0 an integer below 2^24:
// with u = 2^-24, eta = 2^-150 one rounding obeys fl(z) >= z(1-u) - eta for every z >= 0 (half an ulp, normal
// or subnormal), hence e >= fr*LAT*POW*(1-u)^2 - eta*(POW+1) >= fr*lp*(1-2u) - eta*(pmax+1), lp = min LAT*POW.
// The table side (fs_tables.cu) stores lpf <= lp*(1-2^-22) and eta_f >= 2^-149*(pmax+1); here one multiply and one
// subtract, both rounded DOWN, finish it; never negative.  Exactness of the kernel's results does not depend on
// how tight this is, only on its being a lower bound.
__device__ __forceinline__ float fs_energy_lb(float fr, float lpf, float eta_f) {
  const float x = __fsub_rd(__fmul_rd(fr, lpf), eta_f);
  return x > 0.0f ? x : 0.0f;
}

// The shared slot rule (Eq. 1; R:s11), given the two table values.
//   rounds = ceil(q/(beta+1)); t = fl(rounds*lat); e = fl(t*pow)
//   prefill (p==0): ok = fl(wait+t) <= slo;   decode: ok = lat <= slo
struct FsSlot { bool ok; float t, e; };
// the same with the round count already converted (exact: rounds < 2^24)
__device__ __forceinline__ FsSlot fs_slot_f(int p, float lat, float pw, float frounds, float wait, float slo) {
  FsSlot s;
  s.t = __fmul_rn(frounds, lat);
  s.ok = (p == 0) ? (__fadd_rn(wait, s.t) <= slo) : (lat <= slo);
  s.e = __fmul_rn(s.t, pw);
  return s;
}
__device__ __forceinline__ FsSlot fs_slot(int p, float lat, float pw, uint32_t rounds, float wait,
                                          float slo) {
  FsSlot s;
  s.t = __fmul_rn(__uint2float_rn(rounds), lat);
  s.ok = (p == 0) ? (__fadd_rn(wait, s.t) <= slo) : (lat <= slo);
  s.e = __fmul_rn(s.t, pw);
  return s;
}

// ---- mbarrier + 1-D TMA bulk copy (global -> shared), sm_90+ PTX ---------------------------
__device__ __forceinline__ uint32_t fs_smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void fs_mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(fs_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fs_mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fs_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fs_smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void fs_mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(fs_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fs_mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(fs_smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// bytes must be a multiple of 16; src and dst 16-byte aligned
__device__ __forceinline__ void fs_tma_load_1d(void* smem_dst, const void* gsrc, uint32_t bytes,
                                               uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
          "r"(fs_smem_u32(smem_dst)),
      "l"(gsrc), "r"(bytes), "r"(fs_smem_u32(bar))
      : "memory");
}

// ---- counting-sort helper shared by the per-call bucketing passes ---------------------------
// single-block (1,024 threads) inclusive scan of off[1..M] in place (off[0] = 0) and cursor[m] = 0
__device__ __forceinline__ void fs_bucket_scan_block(int32_t* __restrict__ off, int32_t* __restrict__ cursor, int M) {
  __shared__ int32_t part[1024];
  const int t = threadIdx.x, per = (M + 1023) / 1024;
  const int lo = min(M, t * per), hi = min(M, lo + per);
  int32_t sum = 0;
  for (int m = lo; m < hi; ++m) sum += off[m + 1];
  part[t] = sum;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const int32_t add = t >= o ? part[t - o] : 0;
    __syncthreads();
    part[t] += add;
    __syncthreads();
  }
  int32_t acc = part[t] - sum;
  if (t == 0) off[0] = 0;
  for (int m = lo; m < hi; ++m) { acc += off[m + 1]; off[m + 1] = acc; cursor[m] = 0; }
}
