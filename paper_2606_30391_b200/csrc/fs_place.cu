// fs_place.cu — fs_place_batch: global dispatch (§3.3; Eq. 2-3),
// generalised to the (GPU k, grant sigma, frequency phi) grid (R:s2-s6).
//
// For request r and GPU k (eligibility P:195-216):
//   j    = lowest tenant slot with model == m, else cold (needs n_res < 4)
//   wait = T_avail (+ load_ms if cold);  Req_mem = fl(float(L+O)*kv) <= mem_free
//   O    = (21*o_pred+19)/20  (5 % pad; R:s14)
// and for sigma < sm_free, phi < F:
//   dE = fl( fl( A[k][1+j][phi] + fl(e0+e1) ) - Ecur[k] ),  feasible iff co-residents ok (A < INF),
//   fl(wait+t0) <= slo_ttft, LAT1 <= slo_tbt, dE < INF.           (Eq. 2, deadline P:216)
// Result: min over (dE, flat=(k*S+sigma)*F+phi) as ONE 64-bit key (Eq. 3; north_star).
#include "fs_kernels.h"

namespace {

// what a request contributes to every candidate
struct ReqCtx {
  int m; uint32_t L, O; float mem, slo_ttft, slo_tbt, load_ms;
  int br0; uint32_t rounds0; bool valid;
};

__device__ __forceinline__ ReqCtx make_req(const FsView& v, const fs_request& rq) {
  ReqCtx c;
  c.valid = rq.model >= 0 && rq.model < v.d.M && rq.L < (1u << 24) && rq.o_pred < (1u << 24);
  c.m = c.valid ? rq.model : 0; c.L = rq.L; c.O = (21u * rq.o_pred + 19u) / 20u;
  c.mem = __fmul_rn(__uint2float_rn(rq.L + c.O), v.models[c.m].kv_mb_per_token);
  c.slo_ttft = rq.slo_ttft_ms; c.slo_tbt = rq.slo_tbt_ms; c.load_ms = v.models[c.m].load_ms;
  const uint32_t n0 = rq.L < (uint32_t)v.d.B ? rq.L : (uint32_t)v.d.B;   // min(L,B)
  c.br0 = n0 ? (int)n0 - 1 : 0;
  c.rounds0 = n0 ? fs_ceil_div(rq.L, n0) : 0u;
  return c;
}

// what a (request, GPU) pair fixes
struct PairCtx { bool ok; int j, var, br1, smf; float wait, ecur; uint32_t rounds1; };

__device__ __forceinline__ PairCtx make_pair(const FsView& v, const ReqCtx& c, const FsGpuInfo& gi) {
  PairCtx p; p.ok = false; p.j = -1; p.var = 0; p.br1 = 0; p.smf = gi.sm_free; p.wait = 0.f;
  p.ecur = gi.e_cur; p.rounds1 = 0;
  if (gi.n_res < 1 || !(c.mem <= gi.mem_free_mb) || gi.sm_free < 1) return p;
#pragma unroll
  for (int i = FS_RMAX - 1; i >= 0; --i) if (i < gi.n_res && gi.model[i] == c.m) p.j = i;
  if (p.j < 0 && gi.n_res >= FS_RMAX) return p;
  p.wait = gi.t_avail_ms;
  if (p.j < 0) p.wait = __fadd_rn(p.wait, c.load_ms);
  else {
    int b = gi.br1[0];
#pragma unroll
    for (int i = 1; i < FS_RMAX; ++i) if (p.j == i) b = gi.br1[i];
    if (b < 0) return p;
    p.br1 = b;
  }
  p.var = p.j + 1;
  p.rounds1 = fs_ceil_div(c.O, (uint32_t)p.br1 + 1u);
  p.ok = true;
  return p;
}

struct Cand { bool ok; float dE, ttft, tbt; };

// one candidate from the raw planes (used by the generic kernel and by the decode step)
__device__ __forceinline__ Cand eval_cand(const FsView& v, const ReqCtx& c, const PairCtx& p, int k,
                                          int sigma, int phi) {
  const FsDimsDev& d = v.d;
  const size_t o = (size_t)sigma * d.F + phi;
  const size_t i0 = fs_plane(d, c.m, 0, c.br0) + o, i1 = fs_plane(d, c.m, 1, p.br1) + o;
  const float lat1 = v.latT[i1];
  bool ok = true; float t0 = 0.f, e0 = 0.f, e1 = 0.f;
  if (c.L > 0) {
    FsSlot s = fs_slot(0, v.latT[i0], v.powT[i0], c.rounds0, p.wait, c.slo_ttft);
    ok = s.ok; t0 = s.t; e0 = s.e;
  }
  if (c.O > 0) {
    FsSlot s = fs_slot(1, lat1, v.powT[i1], p.rounds1, 0.f, c.slo_tbt);
    ok = ok && s.ok; e1 = s.e;
  }
  const float A = v.gA[((size_t)k * FS_NVAR + p.var) * d.F + phi];
  Cand r;
  r.dE = __fsub_rn(__fadd_rn(A, __fadd_rn(e0, e1)), p.ecur);
  r.ok = ok && (r.dE < FS_INF);            // A == INF (co-residents infeasible) lands here too
  r.ttft = __fadd_rn(p.wait, t0); r.tbt = lat1;
  return r;
}

// ---- generic scorer: any dims, one warp per (request, GPU slice) ---------------------------
__global__ void __launch_bounds__(256) place_generic_kernel(FsView v, int R,
                                                           const fs_request* __restrict__ reqs,
                                                           unsigned long long* __restrict__ keys,
                                                           int nsplit, int kchunk,
                                                           unsigned long long* __restrict__ stats) {
  const int lane = threadIdx.x & 31;
  const long long w = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (w >= (long long)R * nsplit) return;
  const int r = (int)(w / nsplit), part = (int)(w % nsplit);
  const ReqCtx c = make_req(v, reqs[r]);
  if (!c.valid) { if (lane == 0) fs_raise(v.flag, FS_FLAG_REQUEST); return; }
  const FsDimsDev d = v.d;
  const int k0 = part * kchunk, k1 = min(v.K, k0 + kchunk);
  float best = FS_INF; uint32_t bflat = 0xFFFFFFFFu; bool have = false;
  unsigned long long npairs = 0, ncand = 0;
  for (int k = k0; k < k1; ++k) {
    const FsGpuInfo gi = v.ginfo[k];
    const PairCtx p = make_pair(v, c, gi);
    if (!p.ok) continue;
    npairs += 1; ncand += (unsigned long long)p.smf * d.F;
    for (int sg = 0; sg < p.smf; ++sg)
      for (int phi = lane; phi < d.F; phi += 32) {
        const Cand cd = eval_cand(v, c, p, k, sg, phi);
        float dE = cd.dE; if (dE == 0.0f) dE = 0.0f;
        if (cd.ok && (!have || dE < best)) {     // per-lane visiting order is ascending flat
          have = true; best = dE; bflat = (uint32_t)((k * d.S + sg) * d.F + phi);
        }
      }
  }
  unsigned long long key = have ? fs_make_key(best, bflat) : FS_KEY_NONE;
  key = fs_warp_min_key(key);
  if (lane == 0) {
    if (key != FS_KEY_NONE) atomicMin(&keys[r], key);
    if (stats) { atomicAdd(&stats[0], npairs); atomicAdd(&stats[1], ncand); }
  }
}


// =============================================================================================
// Dense scorer for COLD pairs (the request's model is not resident on the GPU), S <= 16, F <= 64.
//
// Factorisation (exact): for a cold pair the decode bucket is 0 and
// the co-resident variant is 0, so everything that depends on (sigma, phi) is per REQUEST:
//   t0[s][f] = fl(rounds0*LAT0)                    er[s][f] = fl(e0 + e1), INF where LAT1 > slo_tbt
// and everything that depends on the GPU is per (k, phi):  A0[k][f], Ecur[k], wait_k, sm_free_k.
// fl(A + x) and fl(x - Ecur) are monotone in x, hence
//   min_s fl(fl(A0 + er[s]) - Ecur) = fl(fl(A0 + min_s er[s]) - Ecur)   over feasible s,
// and fl(wait + t) <= slo  <=>  t <= T*(wait, slo) for the exactly computed threshold T*.
// Per candidate that leaves one compare and one conditional min, on registers.
//
// Layout: one warp = one request, lane owns NPHI adjacent frequencies and all 16 shares
// (2*16*NPHI registers).  A block walks the GPUs in chunks of 32 staged by 1-D TMA bulk copies
// (records + A0 rows) through an mbarrier ring shared by its warps; each lane first evaluates
// eligibility and T* for ONE GPU of the chunk, then the warp sweeps the eligible GPUs.
// The lowest flat index among equal minima is recovered exactly at the end (see below).
// =============================================================================================
constexpr int DENSE_WARPS = 16;
constexpr int DENSE_SMEM_MAX = 200 * 1024;   // of the 227 KB a block may use
constexpr int DENSE_S = 16;

__device__ __forceinline__ uint32_t warp_min_u32(uint32_t x) {
  uint32_t r;
  asm volatile("redux.sync.min.u32 %0, %1, 0xffffffff;" : "=r"(r) : "r"(x));
  return r;
}

// largest t >= 0 with fl(w + t) <= slo, or -1 if there is none.  fl(w + .) is monotone, so the
// answer is characterised by g(T) <= slo < g(nextup(T)); a double-precision guess is verified
// with the fp32 operation itself and a bit-pattern bisection covers whatever it misses.
__device__ __forceinline__ float nextup_nonneg(float x) {       // x >= +0, finite or INF
  return x < FS_INF ? __uint_as_float(__float_as_uint(x) + 1u) : x;
}
__device__ __noinline__ float tstar_bisect(float w, float slo) {
  uint32_t lo = 0u, hi = 0x7F800000u;                            // g(lo) <= slo holds
  if (__fadd_rn(w, FS_INF) <= slo) return FS_INF;
  while (hi - lo > 1u) {
    const uint32_t mid = lo + ((hi - lo) >> 1);
    if (__fadd_rn(w, __uint_as_float(mid)) <= slo) lo = mid; else hi = mid;
  }
  return __uint_as_float(lo);
}
__device__ __forceinline__ float fs_tstar(float w, float slo) {
  if (!(__fadd_rn(w, 0.0f) <= slo)) return -1.0f;                // also NaN
  if (!(slo < FS_INF)) return FS_INF;
  float s = slo; if (s == 0.0f) s = 0.0f;
  const uint32_t sb = __float_as_uint(s);
  const float up = __uint_as_float(s >= 0.0f ? sb + 1u : sb - 1u);   // next float above slo
  const double U = 0.5 * ((double)s + (double)up);               // rounding boundary above slo
  float T = __double2float_rd(U - (double)w);
  if (!(T >= 0.0f)) T = 0.0f;
  if (!(__fadd_rn(w, T) <= slo) && T > 0.0f) T = __uint_as_float(__float_as_uint(T) - 1u);
  const bool ok_here = __fadd_rn(w, T) <= slo;
  const bool ok_next = T < FS_INF && (__fadd_rn(w, nextup_nonneg(T)) <= slo);
  if (ok_here && !ok_next) return T;
  return tstar_bisect(w, slo);
}

// Shared memory of one block: the compact records of its SLICE of the GPUs stay resident for the
// whole kernel (one TMA fill), so the warps never synchronise with each other afterwards.
//   rec [KS]              compact GPU records (32 B each)
//   wb  [DENSE_WARPS][32] per warp: {T*, Ecur, sm_free, GPU} of the chunk being swept
//   bnd [DENSE_WARPS][32] per warp: prefix minima of er / t0 over shares (pruning bounds)
// The A0 rows of the few GPUs that survive the pruning are read through L1/L2.
__host__ __device__ inline size_t dense_smem_bytes(int KS) {
  return (size_t)KS * sizeof(FsGpuRec) + (size_t)DENSE_WARPS * FS_CHUNK * sizeof(float4) +
         (size_t)DENSE_WARPS * 3 * DENSE_S * sizeof(float) + 16;
}

// NPHI adjacent values of row `o` for the lane whose first column is phi0 (columns clamped to the
// row for padded lanes; the caller overrides those); one 64-bit load when the pair is aligned
template <int NPHI>
__device__ __forceinline__ void ld_cols(const float* __restrict__ base, int o, int phi0, int ncol, bool vec,
                                        float (&x)[NPHI]) {
  if (NPHI == 2 && vec) {
    const float2 t = *reinterpret_cast<const float2*>(base + o + min(phi0, ncol - 2));
    x[0] = t.x; x[NPHI - 1] = t.y;
  } else {
#pragma unroll
    for (int i = 0; i < NPHI; ++i) x[i] = base[o + min(phi0 + i, ncol - 1)];
  }
}

template <int NPHI>
__global__ void __launch_bounds__(DENSE_WARPS * 32, 1)
place_dense_kernel(FsView v, int R, const fs_request* __restrict__ reqs,
                   unsigned long long* __restrict__ keys, int nslice, int chunks_per_slice,
                   unsigned int* __restrict__ ctr, const int32_t* __restrict__ warm_off,
                   const FsWarmItem* __restrict__ witems, unsigned long long* __restrict__ stats) {
  extern __shared__ __align__(128) unsigned char dense_smem_raw[];
  constexpr int FT = 32 * NPHI;
  const FsDimsDev d = v.d;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nchunk_all = v.Kpad / FS_CHUNK;
  const int slice = blockIdx.x % nslice;
  const int c0 = slice * chunks_per_slice, c1 = min(nchunk_all, c0 + chunks_per_slice);
  const int nchunk = c1 - c0, KS = nchunk * FS_CHUNK, KSmax = chunks_per_slice * FS_CHUNK;
  FsGpuRec* s_rec = reinterpret_cast<FsGpuRec*>(dense_smem_raw);
  float4* s_wb = reinterpret_cast<float4*>(dense_smem_raw + (size_t)KSmax * sizeof(FsGpuRec));
  float* s_bnd = reinterpret_cast<float*>(s_wb + DENSE_WARPS * FS_CHUNK);   // [warp][2][16] prefix minima
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_bnd + DENSE_WARPS * 3 * DENSE_S);
  const float* gA0 = v.gA0 + (size_t)c0 * FS_CHUNK * FT;   // rows of this slice

  // ---- stage this block's GPU records once: 1-D TMA bulk copies completing on one mbarrier ------
  if (threadIdx.x == 0) { fs_mbar_init(s_bar, 1); fs_mbar_fence_init(); }
  __syncthreads();
  if (threadIdx.x == 0) {
    const uint32_t bytes_rec = (uint32_t)KS * sizeof(FsGpuRec);
    fs_mbar_expect_tx(s_bar, bytes_rec);
    const char* src = reinterpret_cast<const char*>(v.grec + (size_t)c0 * FS_CHUNK);
    char* dst = reinterpret_cast<char*>(s_rec);
    for (uint32_t off = 0; off < bytes_rec; off += 32768u)
      fs_tma_load_1d(dst + off, src + off, min(32768u, bytes_rec - off), s_bar);
  }
  fs_mbar_wait(s_bar, 0);

  float4* wb = s_wb + warp * FS_CHUNK;
  float* bnd = s_bnd + warp * 3 * DENSE_S;      // prefix minima over sigma <= s, all phi, of [0] er (cold), [1] t0, [2] e0
  unsigned long long npairs = 0, ncand = 0, nswept = 0, ncswept = 0, wpairs = 0, wcand = 0, wswept = 0, wcswept = 0;
  const bool vec = NPHI == 2 && (d.F & 1) == 0;
  const int phi0 = lane * NPHI;
  for (;;) {
    // ---- next request of this slice: dynamic, one atomic per warp ----------------------------
    int r = 0;
    if (lane == 0) r = (int)atomicAdd(&ctr[slice], 1u);
    r = __shfl_sync(0xffffffffu, r, 0);
    if (r >= R) break;
    const ReqCtx c = make_req(v, reqs[r]);
    if (!c.valid) { if (lane == 0 && slice == 0) fs_raise(v.flag, FS_FLAG_REQUEST); continue; }
    // ---- phase A: the request's (sigma, phi) tiles in registers -------------------------------
    // L == 0 / O == 0 need no branches: rounds = 0 gives t = e = +0 exactly (tables are finite),
    // and an empty decode slot passes its deadline (threshold +INF).
    float t0[DENSE_S][NPHI], er[DENSE_S][NPHI];
    {
      const float* l0 = v.latT + fs_plane(d, c.m, 0, c.br0); const float* p0 = v.powT + fs_plane(d, c.m, 0, c.br0);
      const float* l1 = v.latT + fs_plane(d, c.m, 1, 0);     const float* p1 = v.powT + fs_plane(d, c.m, 1, 0);
      const float fr0 = __uint2float_rn(c.rounds0), fO = __uint2float_rn(c.O);
      const float tbt = c.O > 0 ? c.slo_tbt : FS_INF;
      uint32_t pe0 = 0x7F800000u;                       // running prefix min of e0 (bits; e0 >= +0)
      __syncwarp();
#pragma unroll
      for (int s4 = 0; s4 < DENSE_S; s4 += 4) {
        float a0[4][NPHI], b0[4][NPHI], a1[4][NPHI], b1[4][NPHI];
#pragma unroll
        for (int u = 0; u < 4; ++u) {                  // 16 independent loads in flight
          const int o = min(s4 + u, d.S - 1) * d.F;
          ld_cols<NPHI>(l0, o, phi0, d.F, vec, a0[u]); ld_cols<NPHI>(p0, o, phi0, d.F, vec, b0[u]);
          ld_cols<NPHI>(l1, o, phi0, d.F, vec, a1[u]); ld_cols<NPHI>(p1, o, phi0, d.F, vec, b1[u]);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          uint32_t ue0 = 0x7F800000u;
#pragma unroll
          for (int i = 0; i < NPHI; ++i) {
            const float tt = __fmul_rn(fr0, a0[u][i]);
            const float e0 = __fmul_rn(tt, b0[u][i]);
            const float ee = __fadd_rn(e0, __fmul_rn(__fmul_rn(fO, a1[u][i]), b1[u][i]));
            const bool in = (s4 + u) < d.S && (phi0 + i) < d.F;
            t0[s4 + u][i] = in ? tt : FS_INF;
            er[s4 + u][i] = (in && a1[u][i] <= tbt) ? ee : FS_INF;
            if (in) ue0 = min(ue0, __float_as_uint(e0));
          }
          pe0 = min(pe0, warp_min_u32(ue0));
          if (lane == 0) bnd[2 * DENSE_S + s4 + u] = __uint_as_float(pe0);
        }
      }
    }
    // ---- bounds for exact pruning: every candidate of a GPU with sm_free = s has
    //   er >= bnd[0][s-1], t0 >= bnd[1][s-1], e0 >= bnd[2][s-1]
    // hence, for a cold pair,  dE >= fl(fl(a_min + bnd[0][s-1]) - Ecur)   (monotone rounding).  er, t0 >= +0, so their bit patterns order like unsigned integers.
    {
      uint32_t pe = 0x7F800000u, pt = 0x7F800000u;
#pragma unroll
      for (int s = 0; s < DENSE_S; ++s) {
        uint32_t ue = 0x7F800000u, ut = 0x7F800000u;
#pragma unroll
        for (int i = 0; i < NPHI; ++i) {
          ue = min(ue, __float_as_uint(er[s][i])); ut = min(ut, __float_as_uint(t0[s][i]));
        }
        pe = min(pe, warp_min_u32(ue)); pt = min(pt, warp_min_u32(ut));
        if (lane == 0) { bnd[s] = __uint_as_float(pe); bnd[DENSE_S + s] = __uint_as_float(pt); }
      }
      __syncwarp();
    }
    float best = FS_INF; int bestk = -1;
    for (int ci = 0; ci < nchunk; ++ci) {
      // best value found so far by any lane (all from GPUs with a lower index than this chunk's)
      const float bestW = fs_unorderable(warp_min_u32(fs_orderable(best)));
      // ---- eligibility + T*: lane <-> one GPU of the chunk ------------------------------------
      const FsGpuRec g = s_rec[ci * FS_CHUNK + lane];
      const int n_res = g.meta & 0xFF, smf = (g.meta >> 8) & 0xFF;
      bool el = n_res >= 1 && n_res < FS_RMAX && smf >= 1 && (c.mem <= g.mem_free_mb);
#pragma unroll
      for (int i = 0; i < FS_RMAX; ++i) el = el && (g.model[i] != c.m);   // resident -> warm path
      float T = -1.0f;
      if (el) {
        npairs += 1; ncand += (unsigned long long)smf * d.F;
        // prune: no candidate of this GPU can beat (or, having a higher index, tie) bestW
        const float lb = __fsub_rn(__fadd_rn(g.a_min, bnd[smf - 1]), g.e_cur);
        if (lb < bestW) {
          T = c.L > 0 ? fs_tstar(__fadd_rn(g.t_avail_ms, c.load_ms), c.slo_ttft) : FS_INF;
          if (!(bnd[DENSE_S + smf - 1] <= T)) T = -1.0f;       // no share meets the TTFT deadline
        }
        if (T >= 0.0f) { nswept += 1; ncswept += (unsigned long long)smf * d.F; }
      }
      // compact the eligible GPUs of the chunk, in ascending order, into the warp's list:
      // {T*, Ecur, sm_free, byte offset of the GPU's A0 row}
      const bool go = el && T >= 0.0f;
      const unsigned mask = __ballot_sync(0xffffffffu, go);
      __syncwarp();
      if (go) wb[__popc(mask & ((1u << lane) - 1u))] =
          make_float4(T, g.e_cur, __int_as_float(smf), __int_as_float(ci * FS_CHUNK + lane));
      __syncwarp();
      const int n_el = __popc(mask);
      // ---- sweep the eligible GPUs of the chunk -------------------------------------------------
      for (int e = 0; e < n_el; ++e) {
        const float4 w = wb[e];
        const float Tst = w.x; const int sfree = __float_as_int(w.z);
        float m[NPHI][2];                               // two min chains per frequency (ILP)
#pragma unroll
        for (int i = 0; i < NPHI; ++i) m[i][0] = m[i][1] = FS_INF;
#define FS_DENSE_STEP(s)                                                              \
  _Pragma("unroll") for (int i = 0; i < NPHI; ++i)                                    \
    asm("{.reg .pred p; setp.le.f32 p, %1, %2; @p min.f32 %0, %0, %3;}"               \
        : "+f"(m[i][(s) & 1]) : "f"(t0[s][i]), "f"(Tst), "f"(er[s][i]));
        switch (sfree) {
          default:
          case 16: FS_DENSE_STEP(15) case 15: FS_DENSE_STEP(14) case 14: FS_DENSE_STEP(13)
          case 13: FS_DENSE_STEP(12) case 12: FS_DENSE_STEP(11) case 11: FS_DENSE_STEP(10)
          case 10: FS_DENSE_STEP(9)  case 9: FS_DENSE_STEP(8)   case 8: FS_DENSE_STEP(7)
          case 7: FS_DENSE_STEP(6)   case 6: FS_DENSE_STEP(5)   case 5: FS_DENSE_STEP(4)
          case 4: FS_DENSE_STEP(3)   case 3: FS_DENSE_STEP(2)   case 2: FS_DENSE_STEP(1)
          case 1: FS_DENSE_STEP(0)
        }
#undef FS_DENSE_STEP
        const int kloc = __float_as_int(w.w);
        float arow[NPHI];
        ld_cols<NPHI>(gA0 + (size_t)kloc * FT, 0, phi0, FT, true, arow);   // rows are FT-padded: aligned
        float x = FS_INF;
#pragma unroll
        for (int i = 0; i < NPHI; ++i) x = fminf(x, __fadd_rn(arow[i], fminf(m[i][0], m[i][1])));
        const float dE = __fsub_rn(x, w.y);          // monotone: min over the lane's phis first
        if (dE < best) { best = dE; bestk = kloc; }
      }
    }
    int bestkg = bestk >= 0 ? c0 * FS_CHUNK + bestk : 0x7FFFFFFF;    // global GPU index of the lane's best
    // ---- warm pairs: GPUs that already host model m (decode bucket, variant and wait depend on
    // the GPU).  Lane <-> item: bound  dE >= fl(fl(a_min + fl(e0min + e1min)) - Ecur)  with
    // e1min = fl(fl(rounds1*l1_min)*p1_min); items that survive are scored candidate by candidate
    // from the planes.  They come after GPUs with a higher index, so ties compare (dE, k) in full
    // and the prune is strict.
    for (int ib = warm_off[c.m]; ib < warm_off[c.m + 1]; ib += 32) {
      uint32_t ordl = 0xFFFFFFFFu; int wk = 0, wsmf = 0;      // orderable bound of the lane's item
      if (ib + lane < warm_off[c.m + 1]) {
        const FsWarmItem it = witems[ib + lane];
        const int kc = it.k / FS_CHUNK;
        if (kc >= c0 && kc < c1 && it.sm_free >= 1 && it.br1 >= 0 && c.mem <= it.mem_free_mb) {
          wpairs += 1; wcand += (unsigned long long)it.sm_free * d.F;
          const float fr1 = __uint2float_rn(fs_ceil_div(c.O, (uint32_t)it.br1 + 1u));
          const float e1lb = __fmul_rn(__fmul_rn(fr1, it.l1_min), it.p1_min);
          const float lb = __fsub_rn(__fadd_rn(it.a_min, __fadd_rn(bnd[2 * DENSE_S + it.sm_free - 1], e1lb)), it.e_cur);
          if (c.O == 0 || it.l1_min <= c.slo_tbt) {
            const float T = c.L > 0 ? fs_tstar(it.t_avail_ms, c.slo_ttft) : FS_INF;
            if (T >= 0.0f && bnd[DENSE_S + it.sm_free - 1] <= T) ordl = fs_orderable(lb);
          }
          wk = it.k; wsmf = it.sm_free;
        }
      }
      // best-first: score the item with the lowest bound, tighten the incumbent, drop every item
      // whose bound is now strictly above it (NaN bounds order above +INF and drop out too)
      for (;;) {
        const uint32_t mn = warp_min_u32(ordl);
        const uint32_t inc = warp_min_u32(fs_orderable(best));
        if (mn == 0xFFFFFFFFu || mn > inc) break;
        const int src = __ffs(__ballot_sync(0xffffffffu, ordl == mn)) - 1;
        if (lane == src) { ordl = 0xFFFFFFFFu; wswept += 1; wcswept += (unsigned long long)wsmf * d.F; }
        const int k = __shfl_sync(0xffffffffu, wk, src);
        const PairCtx p = make_pair(v, c, v.ginfo[k]);
        if (!p.ok) continue;
        for (int sg = 0; sg < p.smf; ++sg)
#pragma unroll
          for (int i = 0; i < NPHI; ++i) {
            const int phi = phi0 + i;
            if (phi < d.F) {
              const Cand cd = eval_cand(v, c, p, k, sg, phi);
              float dE = cd.dE; if (dE == 0.0f) dE = 0.0f;
              if (cd.ok && (dE < best || (dE == best && k < bestkg))) { best = dE; bestkg = k; }
            }
          }
      }
    }
    // ---- recovery: lowest flat index among the lane's candidates that attain its minimum, by the
    // definition (eval_cand), at its best GPU ----------------------------------------------------
    unsigned long long key = FS_KEY_NONE;
    if (bestkg != 0x7FFFFFFF) {
      const PairCtx p = make_pair(v, c, v.ginfo[bestkg]);
      uint32_t flat = 0xFFFFFFFFu;
      for (int sg = 0; sg < p.smf && flat == 0xFFFFFFFFu; ++sg)
#pragma unroll
        for (int i = 0; i < NPHI; ++i) {
          const int phi = phi0 + i;
          if (phi < d.F && flat == 0xFFFFFFFFu) {
            const Cand cd = eval_cand(v, c, p, bestkg, sg, phi);
            if (cd.ok && cd.dE == best) flat = (uint32_t)((bestkg * d.S + sg) * d.F + phi);
          }
        }
      if (flat != 0xFFFFFFFFu) key = fs_make_key(best, flat);
    }
    key = fs_warp_min_key(key);
    if (lane == 0 && key != FS_KEY_NONE) atomicMin(&keys[r], key);
  }
  // work statistics (eligible pairs and their candidates, by the oracle's definition)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    npairs += __shfl_xor_sync(0xffffffffu, npairs, o);
    ncand += __shfl_xor_sync(0xffffffffu, ncand, o);
    nswept += __shfl_xor_sync(0xffffffffu, nswept, o);
    ncswept += __shfl_xor_sync(0xffffffffu, ncswept, o);
    wpairs += __shfl_xor_sync(0xffffffffu, wpairs, o);
    wcand += __shfl_xor_sync(0xffffffffu, wcand, o);
    wswept += __shfl_xor_sync(0xffffffffu, wswept, o);
    wcswept += __shfl_xor_sync(0xffffffffu, wcswept, o);
  }
  if (lane == 0 && stats && (npairs | wpairs)) {
    atomicAdd(&stats[0], npairs); atomicAdd(&stats[1], ncand);
    atomicAdd(&stats[2], wpairs); atomicAdd(&stats[3], wcand);
    atomicAdd(&stats[4], nswept); atomicAdd(&stats[5], ncswept);
    atomicAdd(&stats[6], wswept); atomicAdd(&stats[7], wcswept);
  }
}

// ---- decode: key -> fs_placement (one warp per request, lanes over phi for f_req) ----------
__global__ void __launch_bounds__(256) place_decode_kernel(FsView v, int R,
                                                          const fs_request* __restrict__ reqs,
                                                          const unsigned long long* __restrict__ keys,
                                                          fs_placement* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (r >= R) return;
  const unsigned long long key = keys[r];
  fs_placement o;
  o.gpu = -1; o.sigma = o.phi = o.beta = o.f_req = -1;
  o.energy_mj = o.ttft_ms = o.tbt_ms = FS_INF; o.flat = 0xFFFFFFFFu; o._pad = 0;
  if (key != FS_KEY_NONE) {
    const FsDimsDev d = v.d;
    const uint32_t flat = (uint32_t)key;
    const int phi = flat % d.F, sg = (flat / d.F) % d.S, k = flat / (d.F * d.S);
    const ReqCtx c = make_req(v, reqs[r]);
    const PairCtx p = make_pair(v, c, v.ginfo[k]);
    int f_req = -1;
    for (int base = 0; base < d.F && f_req < 0; base += 32) {
      const int f = base + lane;
      const bool ok = f < d.F && eval_cand(v, c, p, k, sg, f).ok;
      const unsigned m = __ballot_sync(0xffffffffu, ok);
      if (m) f_req = base + __ffs(m) - 1;
    }
    const Cand cd = eval_cand(v, c, p, k, sg, phi);
    o.gpu = k; o.sigma = (int16_t)sg; o.phi = (int16_t)phi; o.beta = (int16_t)p.br1;
    o.f_req = (int16_t)f_req; o.energy_mj = fs_unorderable((uint32_t)(key >> 32));
    o.ttft_ms = cd.ttft; o.tbt_ms = cd.tbt; o.flat = flat;
  }
  if (lane == 0) out[r] = o;
}

}  // namespace

int fsk_place_smem_attr() {
  int e = (int)cudaFuncSetAttribute(place_dense_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, DENSE_SMEM_MAX);
  e |= (int)cudaFuncSetAttribute(place_dense_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, DENSE_SMEM_MAX);
  return e;
}

int fsk_place(const FsView& v, int R, const fs_request* reqs, fs_placement* out,
              const FsPlaceScratch& sc, cudaStream_t st, FsTimers* tm) {
  if (R <= 0) return 0;
  int launches = 0;
  cudaMemsetAsync(sc.keys, 0xFF, sizeof(unsigned long long) * (size_t)R, st);
  cudaMemsetAsync(sc.stats, 0, sizeof(unsigned long long) * 8, st);
  if (v.K <= 0) {
    place_decode_kernel<<<(R + 7) / 8, 256, 0, st>>>(v, R, reqs, sc.keys, out);
    return 1;
  }
  const bool dense_ok = v.d.S <= DENSE_S && v.d.F <= 64 && !sc.force_generic;
  fs_tm_beg(tm, FS_T_PLACE_SCORE, st);
  if (dense_ok) {
    // one persistent block per SM; each holds a slice of the GPUs in shared memory.  The number
    // of slices is what the slice size forces, raised when R alone cannot occupy every SM.
    const int FT = v.d.F <= 32 ? 32 : 64;
    const int nchunk = v.Kpad / FS_CHUNK;
    const size_t fixed = dense_smem_bytes(0), per_chunk = dense_smem_bytes(FS_CHUNK) - fixed;
    const int max_cps = (int)((DENSE_SMEM_MAX - fixed) / per_chunk);
    int nslice = (nchunk + max_cps - 1) / max_cps;
    const int nbatch = (R + DENSE_WARPS - 1) / DENSE_WARPS;
    if (nbatch * nslice < sc.sm_count) nslice = min(nchunk, (sc.sm_count + nbatch - 1) / nbatch);
    const int cps = (nchunk + nslice - 1) / nslice;
    nslice = (nchunk + cps - 1) / cps;
    const int streams = max(1, min(nbatch, sc.sm_count / nslice));
    const int grid = streams * nslice;
    const size_t smem = dense_smem_bytes(cps * FS_CHUNK);
    cudaMemsetAsync(sc.ctr, 0, sizeof(unsigned int) * (size_t)nslice, st);
    if (FT == 32)
      place_dense_kernel<1><<<grid, DENSE_WARPS * 32, smem, st>>>(v, R, reqs, sc.keys, nslice, cps, sc.ctr, sc.warm_off, sc.witems, sc.stats);
    else
      place_dense_kernel<2><<<grid, DENSE_WARPS * 32, smem, st>>>(v, R, reqs, sc.keys, nslice, cps, sc.ctr, sc.warm_off, sc.witems, sc.stats);
    ++launches;
    fs_tm_end(tm, FS_T_PLACE_SCORE, st);
  } else {
    // split the GPUs of one request over several warps when R alone cannot fill the SMs
    const long long want_warps = (long long)sc.sm_count * 32;
    int nsplit = 1;
    if (R < want_warps) nsplit = (int)((want_warps + R - 1) / R);
    if (nsplit > v.K) nsplit = v.K;
    const int kchunk = (v.K + nsplit - 1) / nsplit;
    nsplit = (v.K + kchunk - 1) / kchunk;
    const long long warps = (long long)R * nsplit;
    place_generic_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(v, R, reqs, sc.keys, nsplit,
                                                                     kchunk, sc.stats);
    ++launches;
    fs_tm_end(tm, FS_T_PLACE_SCORE, st);
  }
  fs_tm_beg(tm, FS_T_PLACE_DECODE, st);
  place_decode_kernel<<<(R + 7) / 8, 256, 0, st>>>(v, R, reqs, sc.keys, out);
  fs_tm_end(tm, FS_T_PLACE_DECODE, st);
  ++launches;
  return launches;
}
