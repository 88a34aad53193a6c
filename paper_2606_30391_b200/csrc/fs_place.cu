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

// the same without rounds0 (the caller has a cheaper way to it)
__device__ __forceinline__ ReqCtx make_req_nodiv(const FsView& v, const fs_request& rq) {
  ReqCtx c;
  c.valid = rq.model >= 0 && rq.model < v.d.M && rq.L < (1u << 24) && rq.o_pred < (1u << 24);
  c.m = c.valid ? rq.model : 0; c.L = rq.L; c.O = (21u * rq.o_pred + 19u) / 20u;
  c.mem = __fmul_rn(__uint2float_rn(rq.L + c.O), v.models[c.m].kv_mb_per_token);
  c.slo_ttft = rq.slo_ttft_ms; c.slo_tbt = rq.slo_tbt_ms; c.load_ms = v.models[c.m].load_ms;
  const uint32_t n0 = rq.L < (uint32_t)v.d.B ? rq.L : (uint32_t)v.d.B;   // min(L,B)
  c.br0 = n0 ? (int)n0 - 1 : 0;
  c.rounds0 = 0u;
  return c;
}

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

// one candidate from the raw planes (the decode step)
__device__ __forceinline__ Cand eval_cand(const FsView& v, const ReqCtx& c, const PairCtx& p, int k,
                                          int sigma, int phi) {
  const FsDimsDev& d = v.d;
  const size_t o = (size_t)sigma * d.F + phi;
  const size_t i0 = fs_plane(d, c.m, 0, c.br0) + o, i1 = fs_plane(d, c.m, 1, p.br1) + o;
  const float2 lp0 = v.lpT[i0], lp1 = v.lpT[i1];
  const float lat1 = lp1.x;
  bool ok = true; float t0 = 0.f, e0 = 0.f, e1 = 0.f;
  if (c.L > 0) {
    FsSlot s = fs_slot(0, lp0.x, lp0.y, c.rounds0, p.wait, c.slo_ttft);
    ok = s.ok; t0 = s.t; e0 = s.e;
  }
  if (c.O > 0) {
    FsSlot s = fs_slot(1, lat1, lp1.y, p.rounds1, 0.f, c.slo_tbt);
    ok = ok && s.ok; e1 = s.e;
  }
  const float A = v.gA[((size_t)k * FS_NVAR + p.var) * d.F + phi];
  Cand r;
  r.dE = __fsub_rn(__fadd_rn(A, __fadd_rn(e0, e1)), p.ecur);
  r.ok = ok && (r.dE < FS_INF);            // A == INF (co-residents infeasible) lands here too
  r.ttft = __fadd_rn(p.wait, t0); r.tbt = lat1;
  return r;
}

// =============================================================================================
// Dense scorer, every supported shape (S <= 32; F <= 256 in column blocks of 64): one warp = one request,
// one persistent block per SM, requests handed out by an atomic ticket two requests ahead (the next
// request is already in shared memory, by cp.async, when the current one ends).
//
// Exact factorisation.  For a COLD pair (the request's model is not
// resident on the GPU) the decode bucket is 0 and the co-resident variant is 0, so everything that
// depends on (sigma, phi) is per REQUEST:
//   t0[s][f] = fl(rounds0*LAT0)                    er[s][f] = fl(e0 + e1), INF where LAT1 > slo_tbt
// and everything that depends on the GPU is per (k, phi):  A0[k][f], Ecur[k], wait_k, sm_free_k.
// fl(A + x) and fl(x - Ecur) are monotone in x, hence
//   min_s fl(fl(A0 + er[s]) - Ecur) = fl(fl(A0 + min_s er[s]) - Ecur)   over feasible s,
// and fl(wait + t) <= slo  <=>  t <= T*(wait, slo) for the exactly computed threshold T*.
//
// Per request the warp
//  (a) takes lower bounds on t0, e0 and er over every prefix of shares from the per-plane minima built
//      with the tables (lane <-> share; fs_energy_lb): no table entry is touched for that;
//  (b) scores the WARM pairs (model resident: decode bucket, variant and wait depend on the GPU; listed
//      per model by fs_set_gpu_state), best bound first, candidate by candidate with the definition,
//      straight from the {LAT, POW} planes (two 128-bit loads per share row and lane);
//  (c) only if a cold pair could still win (deadline reachable after the weight load, bound of the best
//      cold-capable GPU not above the incumbent) builds the (sigma, phi) tile {t0, er} in its own
//      shared-memory region - the prefill plane arrives by ONE 1-D TMA bulk copy (cp.async.bulk on the
//      warp's mbarrier; it is contiguous in the plane layout), the decode rows through registers - and
//      walks the cold-capable GPUs in ascending d = a_min - Ecur, lane <-> GPU: eligibility and the exact
//      lower bound fl(fl(a_min + bnd[sm_free]) - Ecur) against the incumbent; the survivors are swept
//      (compare + predicated min per candidate); the walk stops when no later GPU can win;
//  (d) for a cold winner recovers the lowest flat index attaining the minimum from the tile (first candidate
//      in flat order whose definition value equals it), and (one slice) writes the placement record.
// All loops are rolled so that the kernel stays inside the instruction cache.
// =============================================================================================
constexpr int DENSE_MAXW = 20;                // warps per block at most (registers: 65536 / 640 = 102 -> 96)
constexpr int DENSE_SMEM_MAX = 224 * 1024;    // of the 227 KB a block may use

// does any of the four 16-bit models packed in (w0, w1) equal m?  (exact "has a zero halfword" test on the
// XOR; the SIMD-in-a-word video instructions are emulated on this architecture and cost ~30 instructions)
__device__ __forceinline__ bool has_model(uint32_t w0, uint32_t w1, uint32_t mm) {
  const uint32_t x0 = w0 ^ mm, x1 = w1 ^ mm;
  return ((((x0 - 0x00010001u) & ~x0) | ((x1 - 0x00010001u) & ~x1)) & 0x80008000u) != 0u;
}

__device__ __forceinline__ uint32_t warp_min_u32(uint32_t x) { return fs_redux_min_u32(x); }

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

// Shared memory of one block, per warp:  wb [32] {T*, Ecur, sm_free, GPU} of the chunk's survivors, the next
// request (32 B), the warp's mbarrier, 8 work counters, then the tile [S][FT] of {t0, er} pairs (the prefill
// plane {LAT0, POW0} lands there first, by one TMA bulk copy, when the request has cold pairs to sweep).
// The sorted compact GPU records are streamed from global memory (L2) with two 128-bit loads per lane and
// chunk: at pod a request looks at 0.3 chunks.
constexpr int DENSE_WB_OFF = 0, DENSE_REQ_OFF = 512, DENSE_BAR_OFF = 544, DENSE_CNT_OFF = 560, DENSE_TILE_OFF = 640;
__host__ __device__ inline size_t dense_warp_bytes(int S, int FT) {
  return (size_t)DENSE_TILE_OFF + (size_t)S * FT * sizeof(float2);
}
__host__ __device__ inline size_t dense_smem_bytes(int W, int S, int FT) {
  return (size_t)W * dense_warp_bytes(S, FT);
}

// The lane's NPHI adjacent {LAT, POW} entries of a plane row.  Pointers already include the lane's column
// (clamped to the row for padded lanes: they hold copies of the last columns, which no minimum notices,
// and every consumer adds an A row that is +INF there).  VEC: the lane's two entries are one aligned
// 128-bit access (NPHI == 2 and F even): a template parameter, so no branch on the shape at any load.
struct LaneLP { const float2* a; const float2* b; };
template <int NPHI, bool VEC>
__device__ __forceinline__ LaneLP lane_lp(const float2* base, int phi0, int ncol) {
  LaneLP p;
  p.a = base + (NPHI == 2 && VEC ? min(phi0, ncol - 2) : min(phi0, ncol - 1));
  p.b = base + min(phi0 + NPHI - 1, ncol - 1);
  return p;
}
template <int NPHI, bool VEC>
__device__ __forceinline__ void ld_lp(const LaneLP& p, uint32_t o, float (&l)[NPHI], float (&w)[NPHI]) {
  if (NPHI == 2 && VEC) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(p.a + o));
    l[0] = t.x; w[0] = t.y; l[NPHI - 1] = t.z; w[NPHI - 1] = t.w;
  } else {
    const float2 t = __ldg(p.a + o); l[0] = t.x; w[0] = t.y;
    if (NPHI == 2) { const float2 u = __ldg(p.b + o); l[NPHI - 1] = u.x; w[NPHI - 1] = u.y; }
  }
}
// the same from / to the warp's tile (the lane's slot is always aligned)
template <int NPHI>
__device__ __forceinline__ void ld_tile(const float2* p, float (&x)[NPHI], float (&y)[NPHI]) {
  if (NPHI == 2) { const float4 t = *reinterpret_cast<const float4*>(p); x[0] = t.x; y[0] = t.y; x[NPHI - 1] = t.z; y[NPHI - 1] = t.w; }
  else { const float2 t = *p; x[0] = t.x; y[0] = t.y; }
}
template <int NPHI>
__device__ __forceinline__ void st_tile(float2* p, const float (&x)[NPHI], const float (&y)[NPHI]) {
  if (NPHI == 2) *reinterpret_cast<float4*>(p) = make_float4(x[0], y[0], x[NPHI - 1], y[NPHI - 1]);
  else *p = make_float2(x[0], y[0]);
}

// work counters of a counting launch (fs_set_work_stats): per warp in shared memory, flushed per request
enum { ST_CHUNKS = 0, ST_ELIG, ST_SWEPT, ST_CSWEPT, ST_WITEMS, ST_SCORED, ST_CSCORED, ST_REQ, ST_TILES, ST_N };

template <int NPHI, bool VEC, bool COLS>
__global__ void __launch_bounds__(DENSE_MAXW * 32, 1)
place_dense_kernel(FsView v, int R, const fs_request* __restrict__ reqs,
                   unsigned long long* __restrict__ keys, int nslice, int ncb, int chunks_per_slice,
                   unsigned int* __restrict__ ctr, const int32_t* __restrict__ warm_off,
                   const FsWarmItem* __restrict__ witems, unsigned long long* __restrict__ stats,
                   fs_placement* __restrict__ out) {
  extern __shared__ __align__(128) unsigned char dense_smem_raw[];
  constexpr int FT = 32 * NPHI;
  constexpr uint32_t NONE32 = 0xFFFFFFFFu, INFBITS = 0x7F800000u, FULL = 0xffffffffu;
  constexpr int KNONE = 0x7FFFFFFF;
  const FsDimsDev d = v.d;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nchunk_all = v.Kpad / FS_CHUNK;
  const int nsc = COLS ? nslice * ncb : nslice;         // (slice, column block) combinations
  const int sci = blockIdx.x % nsc;
  const int slice = COLS ? sci % nslice : sci;
  const int cb0 = COLS ? (sci / nslice) * 64 : 0;        // first frequency of this block's columns
  const int FA = COLS ? v.FT : FT;                       // row stride of gA0 (F rounded up to 64 when F > 64)
  const int c0 = slice * chunks_per_slice, c1 = min(nchunk_all, c0 + chunks_per_slice);
  const int nchunk = c1 - c0;
  const FsGpuRec* __restrict__ g_rec = v.gsort + (size_t)c0 * FS_CHUNK;     // this block's slice of the SORTED records
  unsigned char* s_warp = dense_smem_raw + (size_t)warp * dense_warp_bytes(d.S, FT);
  float4* wb = reinterpret_cast<float4*>(s_warp + DENSE_WB_OFF);
  fs_request* s_req = reinterpret_cast<fs_request*>(s_warp + DENSE_REQ_OFF);
  uint64_t* w_bar = reinterpret_cast<uint64_t*>(s_warp + DENSE_BAR_OFF);
  uint32_t* s_cnt = reinterpret_cast<uint32_t*>(s_warp + DENSE_CNT_OFF);
  float2* tile = reinterpret_cast<float2*>(s_warp + DENSE_TILE_OFF);
  if (lane == 0) { fs_mbar_init(w_bar, 1); fs_mbar_fence_init(); if (stats) { for (int i = 0; i < ST_N; ++i) s_cnt[i] = 0u; } }
  __syncwarp();

  const double* dsuf = v.dsuf + 1 + c0;
  const double amax = v.dsuf[0];
  const float tmin = (float)v.dsuf[2 + nchunk_all];
  const int phi0 = lane * NPHI;
  const int Fc = d.F - cb0;                              // columns from this block's first one to the end of a row
  const int ncol = min(FT, Fc);                          // columns of this block
  const bool bulk = (d.F & 1) == 0;                      // rows are 16-byte multiples at 16-byte aligned addresses
  const float* a0_lane = v.gA0 + cb0 + phi0;             // rows of gA0 are padded with +INF to FA columns: aligned
  const int ls = min(lane, d.S - 1);                     // lane <-> share for the bounds
  const uint32_t magicB = fs_magic((uint32_t)d.B);
  uint32_t tile_parity = 0;
  // ---- request tickets: r_cur is being scored, r_nxt is on its way into s_req, the ticket after that is
  // requested while r_cur is scored (ticket -> request -> model info would otherwise be a serial chain of
  // three memory latencies at the head of every request)
  const bool req_aligned = (reinterpret_cast<unsigned long long>(reqs) & 15ull) == 0;   // 16-byte copies
  int r_cur = 0, r_nxt = 0;
  if (lane == 0) { r_cur = (int)atomicAdd(&ctr[sci], 1u); r_nxt = (int)atomicAdd(&ctr[sci], 1u); }
  r_cur = __shfl_sync(FULL, r_cur, 0); r_nxt = __shfl_sync(FULL, r_nxt, 0);
  fs_request rq;
  if (r_cur < R) rq = reqs[r_cur];
  while (r_cur < R) {
    const int r = r_cur;
    if (r_nxt < R) {
      const char* src = reinterpret_cast<const char*>(reqs + r_nxt);
      if (req_aligned) {
        if (lane < 2) asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(fs_smem_u32(s_req) + 16u * lane), "l"(src + 16 * lane) : "memory");
      } else if (lane < 8) {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(fs_smem_u32(s_req) + 4u * lane), "l"(src + 4 * lane) : "memory");
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    // the ticket after next: lane 0's atomic writes r_nn in place (predicated, no merge of a branch), and nothing
    // reads it before the volatile shuffle at the end of the request, so the warp never waits for it here
    int r_nn = 0;
    asm volatile("{.reg .pred p; setp.eq.s32 p, %2, 0;\n\t@p atom.global.add.u32 %0, [%1], 1;}"
                 : "+r"(r_nn) : "l"(ctr + sci), "r"(lane) : "memory");
    ReqCtx c = make_req_nodiv(v, rq);
    // rounds0 = ceil(L / min(L, B)): 1 when 0 < L < B, else by multiply-high with the block's constant for B
    c.rounds0 = c.L < (uint32_t)d.B ? (c.L ? 1u : 0u) : fs_ceil_div_magic(c.L, magicB);
    unsigned long long key = FS_KEY_NONE; int kwin = 0;
    // the lane's warm item of this request: GPU, j | br1 << 8 | sm_free << 16 (0: none), rounds1, T_avail, Ecur
    int wk = 0; uint32_t wpk = 0, wr1 = 0; float wta = 0.f, wec = 0.f;
    if (!c.valid) {
      if (lane == 0 && sci == 0) fs_raise(v.flag, FS_FLAG_REQUEST);
    } else {
      // ---- (a) bounds over every prefix of shares (lane <-> share s: shares 0..s, all phi)
      //   b_t0 = min t0 (exact: fl(fr0 * .) is monotone),  b_e0 <= min e0,  b_er <= min er of a cold pair
      const float fr0 = __uint2float_rn(c.rounds0), fO = __uint2float_rn(c.O);
      float b_t0, b_e0, b_er;
      {
        // (32-bit indices: plane index < 2^24, S <= 32)
        const FsPlaneMin pm0 = v.pmin[(uint32_t)(((c.m * 2 + 0) * d.B + c.br0) * d.S + ls)];
        const FsPlaneMin pm1 = v.pmin[(uint32_t)(((c.m * 2 + 1) * d.B + 0) * d.S + ls)];
        b_t0 = __fmul_rn(fr0, pm0.lmin);
        b_e0 = fs_energy_lb(fr0, pm0.lpf, pm0.eta);
        b_er = (c.O == 0 || pm1.lmin <= c.slo_tbt) ? __fadd_rn(b_e0, fs_energy_lb(fO, pm1.lpf, pm1.eta)) : FS_INF;
      }
      const LaneLP q_lp0 = lane_lp<NPHI, VEC>(v.lpT + fs_plane(d, c.m, 0, c.br0) + cb0, phi0, Fc);
      // an empty prefill / decode slot passes its deadline whatever the wait (slot rule, q == 0)
      const float ttft_e = c.L ? c.slo_ttft : FS_INF, tbt_e = c.O ? c.slo_tbt : FS_INF;
      // per-lane incumbent (best, bestk), ordered by (dE, GPU index): the scans are not in index order
      float best = FS_INF; int bestk = KNONE;
      uint32_t bflat = NONE32;   // flat index of the lane's incumbent when the definition body found it (warm pairs)
      // ---- (b) the definition, pair by pair, from the planes: the WARM pairs (GPUs that already host model m),
      // best bound first.
      //   warm bound:  dE >= fl(fl(a_min + fl(b_e0[sm_free-1] + e1lb)) - Ecur),  e1lb = fs_energy_lb(rounds1, ...)
      int ib = warm_off[c.m]; const int ie = warm_off[c.m + 1];
      uint32_t ordl = NONE32;
      bool recover = false; float bestW = FS_INF; uint32_t flat = NONE32;
      for (;;) {
        int k = KNONE;
        int wsrc = -1;                                    // lane that holds the chosen warm item
        while (!recover) {
          const uint32_t mn = warp_min_u32(ordl);
          const uint32_t inc = warp_min_u32(fs_orderable(best));
          if (mn != NONE32 && mn <= inc) {               // best-first: the item with the lowest bound
            const int src = __ffs(__ballot_sync(FULL, ordl == mn)) - 1;
            k = __shfl_sync(FULL, wk, src);
            if (lane == src) ordl = NONE32;
            wsrc = src;
            break;
          }
          if (ib >= ie) {                                 // no item left that could beat the incumbent
            // ---- (c) cold pairs, AFTER the warm ones: a cold start often cannot meet the TTFT deadline at
            // all (load_ms against the SLO), and a warm incumbent lets the scan stop early.  GPUs in ascending
            // d = a_min - Ecur: every candidate of every GPU from chunk ci on has dE >= fl(fl(a + b) - e) with
            // a - e >= dsuf[ci], b >= bmin, a <= amax, and two roundings lose at most 2^-23 (a + b + |a + b - e|);
            // the scan stops as soon as that (with twice the slack) exceeds the incumbent, strictly, so ties
            // still meet every GPU.  No cold pair at all can meet the TTFT deadline if even the earliest
            // T_avail plus the weight load plus the fastest prefill misses it (monotone rounding).
            float bminf = __shfl_sync(FULL, b_er, d.S - 1);
            const float t0min = __shfl_sync(FULL, b_t0, d.S - 1);
            bool cold = bminf < FS_INF && nchunk > 0 &&
                        (c.L == 0 || __fadd_rn(__fadd_rn(tmin, c.load_ms), t0min) <= c.slo_ttft);
            float incW = fs_unorderable(inc);
            if (cold) {                                   // the first chunk's stop test with the table bound
              const double ds = dsuf[0];
              if (!(ds < (double)FS_INF)) cold = false;
              else if (incW < FS_INF) {
                const double x = ds + (double)bminf;
                if (x - 0x1p-22 * (amax + (double)bminf + fabs(x)) - 1e-37 > (double)incW) cold = false;
              }
            }
            if (cold) {
              // ---- the request's tile: {t0, er} per (share, frequency), and the EXACT prefix minima of er
              if (stats && lane == 0) s_cnt[ST_TILES] += 1u;
              const LaneLP q_lp1 = lane_lp<NPHI, VEC>(v.lpT + fs_plane(d, c.m, 1, 0) + cb0, phi0, Fc);
              __syncwarp();
              if (bulk) {
                // generic-proxy accesses of the last request's tile are ordered before the async-proxy writes
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                const float2* src = v.lpT + fs_plane(d, c.m, 0, c.br0) + cb0;
                if (lane == 0) fs_mbar_expect_tx(w_bar, (uint32_t)(d.S * ncol) * 8u);
                __syncwarp();
                if (ncol == FT && d.F == FT) { if (lane == 0) fs_tma_load_1d(tile, src, (uint32_t)(d.S * FT) * 8u, w_bar); }
                else if (lane < d.S) fs_tma_load_1d(tile + lane * FT, src + (size_t)lane * d.F, (uint32_t)ncol * 8u, w_bar);
              } else {
                uint32_t dt = fs_smem_u32(tile + phi0);
                LaneLP g = q_lp0;
                for (int s = 0; s < d.S; ++s) {
                  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dt), "l"(g.a) : "memory");
                  if (NPHI == 2) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dt + 8u), "l"(g.b) : "memory");
                  dt += FT * 8u; g.a += d.F; g.b += d.F;
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
              }
              uint32_t pe = INFBITS;                      // running prefix minimum of er (bits: er >= +0)
              for (int s0 = 0; s0 < d.S; s0 += 4) {
                float a1[4][NPHI], b1[4][NPHI];
#pragma unroll
                for (int u = 0; u < 4; ++u) ld_lp<NPHI, VEC>(q_lp1, (uint32_t)(min(s0 + u, d.S - 1) * d.F), a1[u], b1[u]);
                if (s0 == 0) {                           // the prefill plane has landed in the tile
                  if (bulk) { fs_mbar_wait(w_bar, tile_parity); tile_parity ^= 1u; }
                  else { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
                  __syncwarp();
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                  const int s = s0 + u;
                  if (s < d.S) {
                    float a0[NPHI], b0[NPHI], tt[NPHI], ee[NPHI];
                    ld_tile<NPHI>(tile + s * FT + phi0, a0, b0);
                    uint32_t ue = INFBITS;
#pragma unroll
                    for (int i = 0; i < NPHI; ++i) {
                      const float t = __fmul_rn(fr0, a0[i]);
                      const float e = __fadd_rn(__fmul_rn(t, b0[i]), __fmul_rn(__fmul_rn(fO, a1[u][i]), b1[u][i]));
                      // columns past the row (phi >= F) hold whatever the tile held before: they are masked
                      const bool in = !bulk || phi0 + i < ncol;
                      tt[i] = in ? t : FS_INF;
                      ee[i] = (in && a1[u][i] <= tbt_e) ? e : FS_INF;
                      ue = min(ue, __float_as_uint(ee[i]));
                    }
                    st_tile<NPHI>(tile + s * FT + phi0, tt, ee);
                    pe = min(pe, warp_min_u32(ue));
                    if (lane == s) b_er = __uint_as_float(pe);
                  }
                }
              }
              __syncwarp();
              bminf = __shfl_sync(FULL, b_er, d.S - 1);
              const double bmin = (double)bminf;
              for (int ci = 0; ci < nchunk && bminf < FS_INF; ++ci) {
                incW = fs_unorderable(warp_min_u32(fs_orderable(best)));
                const double ds = dsuf[ci];
                if (!(ds < (double)FS_INF)) break;                 // sentinels only from here on
                if (incW < FS_INF) {
                  const double x = ds + bmin;
                  if (x - 0x1p-22 * (amax + bmin + fabs(x)) - 1e-37 > (double)incW) break;
                }
                // ---- eligibility + bound: lane <-> one GPU of the chunk ---------------------------------
                const FsGpuRec g = g_rec[ci * FS_CHUNK + lane];
                const int smf = (g.meta >> 8) & 0xFF;              // >= 1 (sentinels included)
                const uint32_t mm = (uint32_t)c.m * 0x00010001u;
                const uint32_t* gm = reinterpret_cast<const uint32_t*>(g.model);
                const bool el = (c.mem <= g.mem_free_mb) && !has_model(gm[0], gm[1], mm);
                const float er_lb = __shfl_sync(FULL, b_er, smf - 1), t0_lb = __shfl_sync(FULL, b_t0, smf - 1);
                float T = -1.0f;
                if (el) {
                  // prune: no candidate of this GPU can beat or tie the best found so far
                  const float lb = __fsub_rn(__fadd_rn(g.a_min, er_lb), g.e_cur);
                  if (lb <= incW && lb < FS_INF) {
                    const float wait = __fadd_rn(g.t_avail_ms, c.load_ms);
                    if (c.L == 0) T = FS_INF;
                    else if (__fadd_rn(wait, t0_lb) <= c.slo_ttft) T = fs_tstar(wait, c.slo_ttft);
                  }
                }
                // compact the surviving GPUs of the chunk into the warp's list: {T*, Ecur, sm_free, GPU}
                const bool go = T >= 0.0f;
                const unsigned mask = __ballot_sync(FULL, go);
                if (stats) { const unsigned elm = __ballot_sync(FULL, el); if (lane == 0) { s_cnt[ST_CHUNKS] += 1u; s_cnt[ST_ELIG] += (uint32_t)__popc(elm); } }
                if (mask == 0u) continue;
                __syncwarp();
                if (go) wb[__popc(mask & ((1u << lane) - 1u))] =
                    make_float4(T, g.e_cur, __int_as_float(smf), __int_as_float((int)g.k));
                __syncwarp();
                const int n_el = __popc(mask);
                // ---- sweep the survivors: per candidate one compare and one predicated min ---------------
                for (int e = 0; e < n_el; ++e) {
                  const float4 w = wb[e];
                  const float Tst = w.x; const int sfree = __float_as_int(w.z); const int kk = __float_as_int(w.w);
                  if (stats && lane == 0) { s_cnt[ST_SWEPT] += 1u; s_cnt[ST_CSWEPT] += (uint32_t)(sfree * d.F); }
                  float arow[NPHI], m[NPHI];
                  {
                    const float* ap = a0_lane + (size_t)kk * (size_t)FA;
                    if (NPHI == 2) { const float2 t = *reinterpret_cast<const float2*>(ap); arow[0] = t.x; arow[NPHI - 1] = t.y; }
                    else arow[0] = ap[0];
                  }
#pragma unroll
                  for (int i = 0; i < NPHI; ++i) m[i] = FS_INF;
#pragma unroll 4
                  for (int s = 0; s < sfree; ++s) {
                    float tt[NPHI], ee[NPHI];
                    ld_tile<NPHI>(tile + s * FT + phi0, tt, ee);
#pragma unroll
                    for (int i = 0; i < NPHI; ++i) m[i] = tt[i] <= Tst ? fminf(m[i], ee[i]) : m[i];
                  }
                  float x = FS_INF;
#pragma unroll
                  for (int i = 0; i < NPHI; ++i) x = fminf(x, __fadd_rn(arow[i], m[i]));
                  const float dE = __fsub_rn(x, w.y);          // monotone: min over the lane's phis first
                  if (dE < best || (dE == best && kk < bestk)) { best = dE; bestk = kk; bflat = NONE32; }
                }
              }
            }
            const unsigned long long kq = fs_warp_min_key(((unsigned long long)fs_orderable(best) << 32) | (uint32_t)bestk);
            recover = true; k = (int)(uint32_t)kq; kwin = k; bestW = fs_unorderable((uint32_t)(kq >> 32));
            // a warm winner was scored by the definition in flat order: its lanes already hold their
            // lowest flat index, nothing to recover (a GPU is warm or cold for a request, never both)
            if (k != KNONE && best == bestW && bestk == k) flat = bflat;
            if (__any_sync(FULL, flat != NONE32)) k = KNONE;
            if (k != KNONE) {
              // a COLD winner (it can only come from a sweep, so the tile holds this request's {t0, er}): the lowest
              // flat index attaining the minimum is the first (share, frequency) in flat order whose definition value
              // fl(fl(A0 + er) - Ecur) equals it and whose t0 meets the deadline (t0 <= T*); the same values the
              // definition computes (er = fl(e0 + e1), INF where the TBT deadline fails), read from the tile
              const FsGpuInfo gi = v.ginfo[k];
              const float wait = __fadd_rn(gi.t_avail_ms, c.load_ms);
              const float Tst = c.L == 0 ? FS_INF : fs_tstar(wait, c.slo_ttft);
              float arow[NPHI];
              {
                const float* ap = a0_lane + (size_t)k * (size_t)FA;
                if (NPHI == 2) { const float2 t = *reinterpret_cast<const float2*>(ap); arow[0] = t.x; arow[NPHI - 1] = t.y; }
                else arow[0] = ap[0];
              }
              const uint32_t flat0 = (uint32_t)(k * d.S * d.F + cb0 + phi0);
              for (int s = 0; s < gi.sm_free; ++s) {
                float tt[NPHI], ee[NPHI];
                ld_tile<NPHI>(tile + s * FT + phi0, tt, ee);
                uint32_t f = NONE32;
#pragma unroll
                for (int i = NPHI - 1; i >= 0; --i) {
                  const float dE = __fsub_rn(__fadd_rn(arow[i], ee[i]), gi.e_cur);
                  if (tt[i] <= Tst && dE == bestW) f = flat0 + (uint32_t)(s * d.F + i);
                }
                if (__any_sync(FULL, f != NONE32)) { flat = f; break; }
              }
              k = KNONE;
            }
            break;
          }
          // next 32 items: lane <-> item
          ordl = NONE32;
          const int ix = ib + lane;
          bool have = false; int sidx = 0; float e1lb = 0.f; FsWarmItem it;
          if (ix < ie && (nslice == 1 || ix % nslice == slice)) {
            it = witems[ix];
            if (it.sm_free >= 1 && it.br1 >= 0 && c.mem <= it.mem_free_mb) {
              have = true; sidx = it.sm_free - 1;
              // O = padded output length reaches (21*(2^24-1)+19)/20 > 2^24, past the range in which the
              // multiply-high quotient is exact (fs_common.cuh): such a request (warp-uniform) divides for real
              wr1 = c.O <= (1u << 24) ? fs_ceil_div_magic(c.O, it.magic) : fs_ceil_div(c.O, (uint32_t)it.br1 + 1u);
              e1lb = fs_energy_lb(__uint2float_rn(wr1), it.lp1f, it.eta1);
            }
          }
          const float e0lb = __shfl_sync(FULL, b_e0, sidx), t0lb = __shfl_sync(FULL, b_t0, sidx);
          if (stats) { const uint32_t n = (uint32_t)__popc(__ballot_sync(FULL, have)); if (lane == 0) s_cnt[ST_WITEMS] += n; }
          if (have) {
            const float lb = __fsub_rn(__fadd_rn(it.a_min, __fadd_rn(e0lb, e1lb)), it.e_cur);
            const bool tbt_ok = c.O == 0 || it.l1_min <= c.slo_tbt;
            const bool ttft_ok = c.L == 0 || __fadd_rn(it.t_avail_ms, t0lb) <= c.slo_ttft;
            if (tbt_ok && ttft_ok && lb < FS_INF) ordl = fs_orderable(lb);
            wk = it.k; wpk = (uint32_t)it.j | ((uint32_t)it.br1 << 8) | ((uint32_t)it.sm_free << 16);
            wta = it.t_avail_ms; wec = it.e_cur;
          }
          ib += 32;
        }
        if (k == KNONE) break;                            // no feasible candidate at all, or a warm winner
        // a warm pair's context comes from the item its lane holds (the item passed the memory, bucket and
        // share tests when it was listed): no dependent load of the GPU's summary
        PairCtx p;
        {
          const uint32_t pk = __shfl_sync(FULL, wpk, wsrc);
          p.ok = true; p.j = (int)(pk & 0xFFu); p.var = p.j + 1; p.br1 = (int)((pk >> 8) & 0xFFu); p.smf = (int)(pk >> 16);
          p.wait = __shfl_sync(FULL, wta, wsrc); p.ecur = __shfl_sync(FULL, wec, wsrc);
          p.rounds1 = __shfl_sync(FULL, wr1, wsrc);
        }
        {
          if (stats && lane == 0) { s_cnt[ST_SCORED] += 1u; s_cnt[ST_CSCORED] += (uint32_t)(p.smf * d.F); }
          const LaneLP w_lp1 = lane_lp<NPHI, VEC>(v.lpT + fs_plane(d, c.m, 1, p.br1) + cb0, phi0, Fc);
          const float* Ar = v.gA + ((size_t)k * FS_NVAR + p.var) * d.F + cb0;
          const float fr1 = __uint2float_rn(p.rounds1);
          const float wait_e = c.L ? p.wait : 0.0f;
          float ar[NPHI];
#pragma unroll
          for (int i = 0; i < NPHI; ++i) ar[i] = (phi0 + i) < Fc ? Ar[phi0 + i] : FS_INF;
          // two share rows per stage, software-pipelined: the four plane loads of the NEXT stage are issued
          // before the current one is scored, so a stage's latency hides behind the arithmetic of the one
          // before it.  Each lane keeps the minimum of ITS candidates of this pair and the first (lowest flat)
          // candidate attaining it; merged into the incumbent afterwards.
          float pb = FS_INF; uint32_t pflat = NONE32;
          const uint32_t flat0 = (uint32_t)(k * d.S * d.F + cb0 + phi0);
          float a0[2][2][NPHI], b0[2][2][NPHI], a1[2][2][NPHI], b1[2][2][NPHI];   // [stage buffer][row][phi]
#define FS_BODY_LOAD(BUF, S0)                                                                          \
  _Pragma("unroll") for (int u = 0; u < 2; ++u) {                                                      \
    const uint32_t ro = (uint32_t)(min((S0) + u, p.smf - 1) * d.F);                                    \
    ld_lp<NPHI, VEC>(q_lp0, ro, a0[BUF][u], b0[BUF][u]); ld_lp<NPHI, VEC>(w_lp1, ro, a1[BUF][u], b1[BUF][u]); \
  }
#define FS_BODY_SCORE(BUF, S0)                                                                         \
  _Pragma("unroll") for (int u = 0; u < 2; ++u) {                                                      \
    const int s = (S0) + u;                                                                            \
    _Pragma("unroll") for (int i = 0; i < NPHI; ++i) {                                                 \
      const float t0 = __fmul_rn(fr0, a0[BUF][u][i]);                                                  \
      const float e0 = __fmul_rn(t0, b0[BUF][u][i]);                                                   \
      const float e1 = __fmul_rn(__fmul_rn(fr1, a1[BUF][u][i]), b1[BUF][u][i]);                        \
      const float dE = __fsub_rn(__fadd_rn(ar[i], __fadd_rn(e0, e1)), p.ecur);   /* -0 == +0 in every compare below */ \
      /* rows past sm_free-1 are copies of the last row (clamped loads): the strict '<' below never takes them */ \
      const bool ok = __fadd_rn(wait_e, t0) <= ttft_e && a1[BUF][u][i] <= tbt_e;                       \
      if (ok && dE < pb) { pb = dE; pflat = flat0 + (uint32_t)(s * d.F + i); }   /* INF never enters */ \
    }                                                                                                  \
  }
          FS_BODY_LOAD(0, 0)
#pragma unroll 1
          for (int s4 = 0; s4 < p.smf; s4 += 4) {
            FS_BODY_LOAD(1, s4 + 2)
            FS_BODY_SCORE(0, s4)
            if (s4 + 2 >= p.smf) break;
            FS_BODY_LOAD(0, s4 + 4)
            FS_BODY_SCORE(1, s4 + 2)
          }
#undef FS_BODY_LOAD
#undef FS_BODY_SCORE
          if (pb < best || (pb == best && k < bestk)) { best = pb; bestk = k; bflat = pflat; }
        }
      }
      key = flat != NONE32 ? fs_make_key(bestW, flat) : FS_KEY_NONE;
      key = fs_warp_min_key(key);
    }
    if (COLS || out == nullptr) {                      // several slices / column blocks: merge by key, decode afterwards
      if (lane == 0 && key != FS_KEY_NONE) atomicMin(&keys[r], key);
    } else {
      // one slice: this warp saw every GPU, so it writes the placement record itself: the chosen
      // share row is evaluated once more across phi by the definition for f_req (lowest feasible
      // phi of the chosen (GPU, share)) and the chosen candidate's TTFT / TBT
      fs_placement o; o.gpu = -1; o.sigma = o.phi = o.beta = o.f_req = -1;
      o.energy_mj = o.ttft_ms = o.tbt_ms = FS_INF; o.flat = 0xFFFFFFFFu; o._pad = 0;
      if (key != FS_KEY_NONE) {
        const uint32_t fl = (uint32_t)key;
        // the winning GPU is known (kwin); one small division instead of three 32-bit ones
        const int ks = kwin, rem = (int)(fl - (uint32_t)(ks * d.S * d.F)), sgs = rem / d.F, phis = rem - sgs * d.F;
        // a warm winner's context is still in the lane that holds its list item (a GPU is listed once per model);
        // only a cold winner reads the GPU's summary
        PairCtx p;
        const unsigned hit = __ballot_sync(FULL, wpk != 0u && wk == ks);
        if (hit) {
          const int src = __ffs(hit) - 1;
          const uint32_t pk = __shfl_sync(FULL, wpk, src);
          p.ok = true; p.j = (int)(pk & 0xFFu); p.var = p.j + 1; p.br1 = (int)((pk >> 8) & 0xFFu); p.smf = (int)(pk >> 16);
          p.wait = __shfl_sync(FULL, wta, src); p.ecur = __shfl_sync(FULL, wec, src);
          p.rounds1 = __shfl_sync(FULL, wr1, src);
        } else {
          p = make_pair(v, c, v.ginfo[ks]);
        }
        const LaneLP q0 = lane_lp<NPHI, VEC>(v.lpT + fs_plane(d, c.m, 0, c.br0), phi0, d.F);
        const LaneLP q1 = lane_lp<NPHI, VEC>(v.lpT + fs_plane(d, c.m, 1, p.br1), phi0, d.F);
        const float* Ar = v.gA + ((size_t)ks * FS_NVAR + p.var) * d.F;
        const float fr0 = __uint2float_rn(c.rounds0), fr1 = __uint2float_rn(p.rounds1);
        float a0[NPHI], b0[NPHI], a1[NPHI], b1[NPHI];
        const uint32_t ro = (uint32_t)(sgs * d.F);
        ld_lp<NPHI, VEC>(q0, ro, a0, b0); ld_lp<NPHI, VEC>(q1, ro, a1, b1);
        uint32_t fmin = NONE32; float ttft = 0.0f, tbt = 0.0f;
#pragma unroll
        for (int i = 0; i < NPHI; ++i) {
          const int phi = phi0 + i;
          const float ar = phi < d.F ? Ar[phi] : FS_INF;
          const float t0 = __fmul_rn(fr0, a0[i]);
          const float dE = __fsub_rn(__fadd_rn(ar, __fadd_rn(__fmul_rn(t0, b0[i]), __fmul_rn(__fmul_rn(fr1, a1[i]), b1[i]))), p.ecur);
          const bool ok = (c.L == 0 || __fadd_rn(p.wait, t0) <= c.slo_ttft) && (c.O == 0 || a1[i] <= c.slo_tbt) && dE < FS_INF;
          if (ok) fmin = min(fmin, (uint32_t)phi);
          if (phi == phis) { ttft = __fadd_rn(p.wait, t0); tbt = a1[i]; }
        }
        fmin = warp_min_u32(fmin);
        const int owner = phis / NPHI;
        ttft = __shfl_sync(FULL, ttft, owner); tbt = __shfl_sync(FULL, tbt, owner);
        o.gpu = ks; o.sigma = (int16_t)sgs; o.phi = (int16_t)phis; o.beta = (int16_t)p.br1;
        o.f_req = (int16_t)(int)fmin; o.energy_mj = fs_unorderable((uint32_t)(key >> 32));
        o.ttft_ms = ttft; o.tbt_ms = tbt; o.flat = fl;
      }
      if (lane == 0) out[r] = o;
    }
    if (stats) {
      __syncwarp();
      if (lane < ST_N) { const uint32_t x = lane == ST_REQ ? 1u : s_cnt[lane]; if (x) atomicAdd(&stats[lane], (unsigned long long)x); s_cnt[lane] = 0u; }
      __syncwarp();
    }
    // ---- advance: the next request has landed in s_req
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();
    if (r_nxt < R) rq = *s_req;
    __syncwarp();
    r_cur = r_nxt;
    asm volatile("shfl.sync.idx.b32 %0, %1, 0, 31, 0xffffffff;" : "=r"(r_nxt) : "r"(r_nn) : "memory");
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

// =============================================================================================
// fs_dispatch: the paper's own three-phase dispatcher (Fig. 6), ONE operating point
// per GPU: S_k = SM_free (sigma = sm_free-1), f_k = F_curr.
//   Phase 1 feasibility at F_curr;  Phase 2 (Eq. 2-3) E^k = Power x Latency
//   of the request's own work, argmin; 2 % band -> most free memory, largest SM_free, lowest k
//   (P:229);  Phase 3 F_max retry, first feasible GPU in T_avail order; then scale-out:
//   energy-optimal feasible frequency of a fresh GPU (all S units, wait = load_ms).
// One warp = one request.  The warp builds the request's (sigma, phi) tiles t0 / er for the cold
// case in shared memory once (as the S x F scorer does); a cold (request, GPU) pair is then two
// shared-memory reads at (sm_free-1, F_curr), a warm pair (model resident: its own decode bucket)
// reads the planes.  Lanes <-> GPUs; reductions by redux / 64-bit key shuffles.
// =============================================================================================
constexpr int DISP_WARPS = 8;
constexpr int DISP_NC = 4;                    // group minima kept per lane: GPUs beyond 32*32*DISP_GC*DISP_NC are always revisited
constexpr int DISP_GC = 4;                    // chunks of 32 GPUs per group (one reduction, DISP_GC loads in flight)

struct OwnEval { bool ok; float e, ttft, tbt; };

// the request's own prefill + decode work at (phi, sg) on pair p, from the planes (definition)
// the same from the four table entries (l0, p0: prefill; l1, p1: decode)
__device__ __forceinline__ OwnEval own_eval_vals(const ReqCtx& c, uint32_t rounds1, float wait, float l0, float p0,
                                                 float l1, float p1) {
  bool ok = true; float t0 = 0.f, e0 = 0.f, e1 = 0.f;
  if (c.L > 0) { FsSlot s = fs_slot(0, l0, p0, c.rounds0, wait, c.slo_ttft); ok = s.ok; t0 = s.t; e0 = s.e; }
  if (c.O > 0) { FsSlot s = fs_slot(1, l1, p1, rounds1, 0.f, c.slo_tbt); ok = ok && s.ok; e1 = s.e; }
  OwnEval r; r.e = __fadd_rn(e0, e1); r.ok = ok && r.e < FS_INF;
  r.ttft = __fadd_rn(wait, t0); r.tbt = l1;
  return r;
}
__device__ __forceinline__ OwnEval own_eval_planes(const FsView& v, const ReqCtx& c, int br1, uint32_t rounds1,
                                                   float wait, int sg, int phi) {
  const FsDimsDev& d = v.d;
  const size_t o = (size_t)sg * d.F + phi;
  const size_t i0 = fs_plane(d, c.m, 0, c.br0) + o, i1 = fs_plane(d, c.m, 1, br1) + o;
  const float2 a = v.lpT[i0], b = v.lpT[i1];
  return own_eval_vals(c, rounds1, wait, a.x, a.y, b.x, b.y);
}

struct DispPair { bool ok; float e; };
// pair (request, GPU k with compact record g) at frequency phi (< 0: the GPU's F_curr).  Cold pairs
// (model not resident: two packed 16-bit compares) read the tiles; warm pairs and the no-tile case
// go through the full summary, make_pair and the planes.
__device__ __forceinline__ DispPair disp_pair(const FsView& v, const ReqCtx& c, const FsGpuRec& g, int k, int phi,
                                              const float* tl_t0, const float* tl_er, int FT) {
  DispPair r; r.ok = false; r.e = FS_INF;
  const int n_res = g.meta & 0xFF, smf = (g.meta >> 8) & 0xFF;
  if (phi < 0) phi = (g.meta >> 16) & 0xFFFF;
  if (n_res < 1 || smf < 1 || !(c.mem <= g.mem_free_mb)) return r;
  const uint32_t mm = (uint32_t)c.m * 0x00010001u;
  const uint32_t* gm = reinterpret_cast<const uint32_t*>(g.model);
  if (tl_t0) {
    // resident model: a WARM pair, scored from the per-model list instead (a rare lane would make
    // the whole warp take the slow path in almost every chunk)
    if (has_model(gm[0], gm[1], mm) || n_res >= FS_RMAX) return r;
    const int o = (smf - 1) * FT + phi;
    r.e = tl_er[o];
    r.ok = (c.L == 0 || __fadd_rn(__fadd_rn(g.t_avail_ms, c.load_ms), tl_t0[o]) <= c.slo_ttft) && r.e < FS_INF;
    return r;
  }
  const PairCtx p = make_pair(v, c, v.ginfo[k]);
  if (!p.ok) return r;
  const OwnEval ev = own_eval_planes(v, c, p.br1, p.rounds1, p.wait, p.smf - 1, phi);
  r.ok = ev.ok; r.e = ev.e;
  return r;
}

// warm pair from the per-model list (phi < 0: the GPU's F_curr)
__device__ __forceinline__ DispPair disp_warm(const FsView& v, const ReqCtx& c, const FsWarmItem& it, int phi) {
  DispPair r; r.ok = false; r.e = FS_INF;
  // the item carries what make_pair would read from the GPU's summary (listed items have n_res >= 1 and host
  // the model in slot j): no dependent load before the table entries are requested
  if (it.sm_free < 1 || it.br1 < 0 || !(c.mem <= it.mem_free_mb)) return r;
  const OwnEval ev = own_eval_planes(v, c, it.br1, fs_ceil_div(c.O, (uint32_t)it.br1 + 1u), it.t_avail_ms,
                                     it.sm_free - 1, phi < 0 ? it.f_cur : phi);
  r.ok = ev.ok; r.e = ev.e;
  return r;
}

// reductions over the warps that share a request: the warp alone, or (BLOCK) all DISP_WARPS warps of the block
template <bool BLOCK>
__device__ __forceinline__ uint32_t disp_min_u32(uint32_t x, uint32_t* s_red, int warp, int lane) {
  x = warp_min_u32(x);
  if (BLOCK) {
    __syncthreads();
    if (lane == 0) s_red[warp] = x;
    __syncthreads();
    x = s_red[0];
#pragma unroll
    for (int w = 1; w < DISP_WARPS; ++w) x = min(x, s_red[w]);
  }
  return x;
}
template <bool BLOCK>
__device__ __forceinline__ unsigned long long disp_min_key(unsigned long long k, unsigned long long* s_red, int warp, int lane) {
  k = fs_warp_min_key(k);
  if (BLOCK) {
    __syncthreads();
    if (lane == 0) s_red[warp] = k;
    __syncthreads();
    k = s_red[0];
#pragma unroll
    for (int w = 1; w < DISP_WARPS; ++w) k = s_red[w] < k ? s_red[w] : k;
  }
  return k;
}

// BLOCK = false: one warp per request (batches).  BLOCK = true: one block per request, its warps split
// the GPUs (few requests, e.g. a single arrival against thousands of GPUs: the scan is the latency).
template <int NPHI, bool BLOCK>
__global__ void __launch_bounds__(DISP_WARPS * 32) dispatch_kernel(FsView v, int R,
                                                                  const fs_request* __restrict__ reqs,
                                                                  fs_placement* __restrict__ out, int use_tiles,
                                                                  const int32_t* __restrict__ warm_off,
                                                                  const FsWarmItem* __restrict__ witems) {
  extern __shared__ __align__(16) unsigned char disp_smem[];
  __shared__ unsigned long long s_red[DISP_WARPS];
  uint32_t* s_red32 = reinterpret_cast<uint32_t*>(s_red);
  constexpr int FT = 32 * NPHI;
  constexpr int NW = BLOCK ? DISP_WARPS : 1;           // warps per request
  const FsDimsDev d = v.d;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int sub = BLOCK ? warp : 0;
  const int r = BLOCK ? (int)blockIdx.x : (int)blockIdx.x * DISP_WARPS + warp;
  if (r >= R) return;
  // F > 64: no tiles, every pair from the planes
  float* tl_t0 = use_tiles ? reinterpret_cast<float*>(disp_smem) + (size_t)(BLOCK ? 0 : warp) * 2 * d.S * FT : nullptr;
  float* tl_er = tl_t0 + d.S * FT;
  fs_placement o;
  o.gpu = -1; o.sigma = o.phi = o.beta = o.f_req = -1;
  o.energy_mj = o.ttft_ms = o.tbt_ms = FS_INF; o.flat = 0xFFFFFFFFu; o._pad = 0;
  const ReqCtx c = make_req(v, reqs[r]);
  if (!c.valid) { if (lane == 0 && sub == 0) { fs_raise(v.flag, FS_FLAG_REQUEST); out[r] = o; } return; }
  // ---- the request's cold tiles: t0 = fl(rounds0*LAT0), er = fl(e0 + e1) (INF where LAT1 > slo_tbt)
  if (use_tiles) {
    const float2* lp0 = v.lpT + fs_plane(d, c.m, 0, c.br0);   // {LAT, POW} planes: prefill bucket, decode bucket 0
    const float2* lp1 = v.lpT + fs_plane(d, c.m, 1, 0);
    const float fr0 = __uint2float_rn(c.rounds0), fO = __uint2float_rn(c.O);
    const float tbt = c.O > 0 ? c.slo_tbt : FS_INF;
    const int phi0 = lane * NPHI;
#pragma unroll 2
    for (int s = sub; s < d.S; s += NW) {
      const int ofs = s * d.F;
#pragma unroll
      for (int i = 0; i < NPHI; ++i) {
        const bool in = (phi0 + i) < d.F;
        const int col = min(phi0 + i, d.F - 1);
        const float2 x0 = lp0[ofs + col], x1 = lp1[ofs + col];
        const float t = __fmul_rn(fr0, x0.x);
        const float e = __fadd_rn(__fmul_rn(t, x0.y), __fmul_rn(__fmul_rn(fO, x1.x), x1.y));
        tl_t0[s * FT + phi0 + i] = in ? t : FS_INF;
        tl_er[s * FT + phi0 + i] = (in && x1.x <= tbt) ? e : FS_INF;
      }
    }
    if (BLOCK) __syncthreads(); else __syncwarp();
  }
  // ---- Phase 1 + 2 at F_curr: E_min, then the 2 % band with the stability tie-breaker ----------
  // This warp's chunks of 32 GPUs: sub, sub + NW, ..., taken DISP_GC at a time; lane j of cmin keeps the
  // minimum of the warp's j-th group so that the band scan only revisits groups that hold a candidate
  // inside the band.  grec is padded to a multiple of 32 records (n_res = 0).
  const int nchunk = v.Kpad / 32;
  uint32_t emin_o = 0xFFFFFFFFu, cmin[DISP_NC];
#pragma unroll
  for (int u = 0; u < DISP_NC; ++u) cmin[u] = 0xFFFFFFFFu;
  for (int j0 = 0; sub + j0 * NW < nchunk; j0 += DISP_GC) {
    FsGpuRec g4[DISP_GC];                              // DISP_GC independent record loads in flight
#pragma unroll
    for (int u = 0; u < DISP_GC; ++u) {
      const int ch = sub + (j0 + u) * NW;
      g4[u] = v.grec[min(ch, nchunk - 1) * 32 + lane];
      if (ch >= nchunk) g4[u].meta = 0u;               // past the end: n_res = 0, never a candidate
    }
    uint32_t eo = 0xFFFFFFFFu;
#pragma unroll
    for (int u = 0; u < DISP_GC; ++u) {
      const DispPair dp = disp_pair(v, c, g4[u], (sub + (j0 + u) * NW) * 32 + lane, -1, tl_t0, tl_er, FT);
      if (dp.ok) eo = min(eo, fs_orderable(dp.e));
    }
    const uint32_t cm = warp_min_u32(eo);
    const int gj = j0 / DISP_GC;
#pragma unroll
    for (int u = 0; u < DISP_NC; ++u) if ((gj >> 5) == u && (gj & 31) == lane) cmin[u] = cm;
    emin_o = min(emin_o, cm);
  }
  // no GPUs (K = 0): the warm lists were not rebuilt for this state (they may hold the previous poll's items, or
  // nothing at all on a fresh context) and must not be read
  const bool warm = use_tiles && v.K > 0;
  const int wb0 = warm ? warm_off[c.m] : 0, wb1 = warm ? warm_off[c.m + 1] : 0;
  for (int ib = wb0 + sub * 32; ib < wb1; ib += 32 * NW) {
    uint32_t eo = 0xFFFFFFFFu;
    if (ib + lane < wb1) {
      const DispPair dp = disp_warm(v, c, witems[ib + lane], -1);
      if (dp.ok) eo = fs_orderable(dp.e);
    }
    emin_o = min(emin_o, warp_min_u32(eo));
  }
  emin_o = disp_min_u32<BLOCK>(emin_o, s_red32, warp, lane);
  int phase = -1, kbest = -1, phibest = -1;
  if (emin_o != 0xFFFFFFFFu) {
    const float band = __fmul_rn(1.02f, fs_unorderable(emin_o));
    const uint32_t band_o = fs_orderable(band);
    unsigned long long key = FS_KEY_NONE;              // (most memory, largest SM_free, lowest k)
    for (int j0 = 0; sub + j0 * NW < nchunk; j0 += DISP_GC) {
      const int gj = j0 / DISP_GC;
      if (gj < 32 * DISP_NC) {
        uint32_t cm = 0xFFFFFFFFu;
#pragma unroll
        for (int u = 0; u < DISP_NC; ++u) if ((gj >> 5) == u) cm = cmin[u];
        cm = __shfl_sync(0xffffffffu, cm, gj & 31);
        if (cm > band_o) continue;                     // no candidate of this group is inside the band
      }
      for (int u = 0; u < DISP_GC; ++u) {
        const int ch = sub + (j0 + u) * NW;
        if (ch >= nchunk) break;
        const int k = ch * 32 + lane;
        const FsGpuRec g = v.grec[k];
        const DispPair dp = disp_pair(v, c, g, k, -1, tl_t0, tl_er, FT);
        if (dp.ok && dp.e <= band) {
          const unsigned long long kk = ((unsigned long long)(~fs_orderable(g.mem_free_mb)) << 32) |
                                        ((unsigned long long)(uint32_t)(d.S - (int)((g.meta >> 8) & 0xFF)) << 24) | (uint32_t)k;
          key = kk < key ? kk : key;
        }
      }
    }
    for (int ib = wb0 + sub * 32 + lane; ib < wb1; ib += 32 * NW) {
      const FsWarmItem it = witems[ib];
      const DispPair dp = disp_warm(v, c, it, -1);
      if (dp.ok && dp.e <= band) {
        const unsigned long long kk = ((unsigned long long)(~fs_orderable(it.mem_free_mb)) << 32) |
                                      ((unsigned long long)(uint32_t)(d.S - it.sm_free) << 24) | (uint32_t)it.k;
        key = kk < key ? kk : key;
      }
    }
    key = disp_min_key<BLOCK>(key, s_red, warp, lane);
    kbest = (int)((uint32_t)key & 0xFFFFFFu); phase = 1;
    phibest = v.ginfo[kbest].f_cur;
  } else {
    // ---- Phase 3: F_max retry, first feasible GPU in T_avail order ------------------------------
    unsigned long long key = FS_KEY_NONE;
    for (int ch = sub; ch < nchunk; ch += NW) {
      const int k = ch * 32 + lane;
      const FsGpuRec g = v.grec[k];
      const DispPair dp = disp_pair(v, c, g, k, d.F - 1, tl_t0, tl_er, FT);
      if (dp.ok) {
        const unsigned long long kk = ((unsigned long long)fs_orderable(g.t_avail_ms) << 32) | (uint32_t)k;
        key = kk < key ? kk : key;
      }
    }
    for (int ib = wb0 + sub * 32 + lane; ib < wb1; ib += 32 * NW) {
      const FsWarmItem it = witems[ib];
      const DispPair dp = disp_warm(v, c, it, d.F - 1);
      if (dp.ok) {
        const unsigned long long kk = ((unsigned long long)fs_orderable(it.t_avail_ms) << 32) | (uint32_t)it.k;
        key = kk < key ? kk : key;
      }
    }
    key = disp_min_key<BLOCK>(key, s_red, warp, lane);
    if (key != FS_KEY_NONE) { kbest = (int)(uint32_t)key; phase = 2; phibest = d.F - 1; }
  }
  if (sub != 0) return;                                // the request's first warp writes the record
  if (kbest >= 0) {
    const PairCtx p = make_pair(v, c, v.ginfo[kbest]);
    const OwnEval ev = own_eval_planes(v, c, p.br1, p.rounds1, p.wait, p.smf - 1, phibest);
    o.gpu = kbest; o.sigma = (int16_t)(p.smf - 1); o.phi = (int16_t)phibest; o.beta = (int16_t)p.br1;
    o.f_req = (int16_t)phase; o.energy_mj = ev.e; o.ttft_ms = ev.ttft; o.tbt_ms = ev.tbt;
    o.flat = (uint32_t)((kbest * d.S + p.smf - 1) * d.F + phibest);
  } else {
    // ---- scale-out: energy-optimal feasible frequency of a fresh GPU (all S units, wait = load_ms)
    unsigned long long key = FS_KEY_NONE;
    for (int phi = lane; phi < d.F; phi += 32) {
      bool ok; float e;
      if (use_tiles) {
        const float t0 = tl_t0[(d.S - 1) * FT + phi]; e = tl_er[(d.S - 1) * FT + phi];
        ok = (c.L == 0 || __fadd_rn(c.load_ms, t0) <= c.slo_ttft) && e < FS_INF;
      } else { const OwnEval ev = own_eval_planes(v, c, 0, c.O, c.load_ms, d.S - 1, phi); ok = ev.ok; e = ev.e; }
      if (ok) {
        const unsigned long long kk = fs_make_key(e, (uint32_t)phi);
        key = kk < key ? kk : key;
      }
    }
    key = fs_warp_min_key(key);
    if (key != FS_KEY_NONE) {
      const int phi = (int)(uint32_t)key;
      const OwnEval ev = own_eval_planes(v, c, 0, c.O, c.load_ms, d.S - 1, phi);
      o.sigma = (int16_t)(d.S - 1); o.phi = (int16_t)phi; o.beta = 0; o.f_req = 3;
      o.energy_mj = ev.e; o.ttft_ms = ev.ttft; o.tbt_ms = ev.tbt;
    }
  }
  if (lane == 0) out[r] = o;
}

// ---------------------------------------------------------------------------------------------------
// fs_dispatch_commit: the dispatcher with the sequential commit pass between the requests of one batch
// (the rest of NEXT-2; reading R:s34 of P:214-218).  The requests are inherently
// serial (request r sees the records request r-1 left), so ONE block walks them in order; the parallel
// axis is the GPUs: thread t owns GPUs t, t + blockDim, ... and is the only reader and writer of their
// mutable record work[k] = (T_avail, free memory, F_curr).  Per request: one block-wide minimum for
// E_min, one for the band's stability key (or the F_max retry's T_avail key); the owner of the winner
// writes the decision and commits it.  Reductions alternate between two shared buffers: one barrier each.
constexpr int CM_THREADS = 1024;

__device__ __forceinline__ unsigned long long cm_block_min(unsigned long long x, unsigned long long (*buf)[CM_THREADS / 32],
                                                           int& par, int nwarp, int warp, int lane) {
  x = fs_warp_min_key(x);
  if (lane == 0) buf[par][warp] = x;
  __syncthreads();
  unsigned long long y = lane < nwarp ? buf[par][lane] : FS_KEY_NONE;
  par ^= 1;
  return fs_warp_min_key(y);
}

struct CmEval { bool ok; PairCtx p; OwnEval ev; };
// GPU k as the records stand now, at frequency phi (< 0: its F_curr)
__device__ __forceinline__ CmEval cm_eval(const FsView& v, const ReqCtx& c, int k, const fs_gpu_avail& w, int phi) {
  FsGpuInfo gi = v.ginfo[k];
  gi.t_avail_ms = w.t_avail_ms; gi.mem_free_mb = w.mem_free_mb; gi.f_cur = w.f_cur;
  CmEval r; r.p = make_pair(v, c, gi); r.ok = false;
  if (!r.p.ok) return r;
  r.ev = own_eval_planes(v, c, r.p.br1, r.p.rounds1, r.p.wait, r.p.smf - 1, phi < 0 ? gi.f_cur : phi);
  r.ok = r.ev.ok;
  return r;
}

__global__ void __launch_bounds__(CM_THREADS) dispatch_commit_kernel(FsView v, int R,
                                                                     const fs_request* __restrict__ reqs,
                                                                     fs_placement* __restrict__ out,
                                                                     fs_gpu_avail* __restrict__ work) {
  __shared__ unsigned long long s_buf[2][CM_THREADS / 32];
  const FsDimsDev d = v.d;
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
  int par = 0;
  for (int k = tid; k < v.K; k += nthr) {
    const FsGpuInfo gi = v.ginfo[k];
    fs_gpu_avail w; w.t_avail_ms = gi.t_avail_ms; w.mem_free_mb = gi.mem_free_mb; w.f_cur = gi.f_cur; w._pad = 0;
    work[k] = w;
  }
  for (int r = 0; r < R; ++r) {
    fs_placement o;
    o.gpu = -1; o.sigma = o.phi = o.beta = o.f_req = -1;
    o.energy_mj = o.ttft_ms = o.tbt_ms = FS_INF; o.flat = 0xFFFFFFFFu; o._pad = 0;
    const ReqCtx c = make_req(v, reqs[r]);
    if (!c.valid) { if (tid == 0) { fs_raise(v.flag, FS_FLAG_REQUEST); out[r] = o; } continue; }
    // ---- Phase 1 + 2 at F_curr: E_min over the feasible GPUs ------------------------------------
    unsigned long long key = FS_KEY_NONE;
    for (int k = tid; k < v.K; k += nthr) {
      const CmEval e = cm_eval(v, c, k, work[k], -1);
      if (e.ok) { const unsigned long long kk = fs_orderable(e.ev.e); key = kk < key ? kk : key; }
    }
    key = cm_block_min(key, s_buf, par, nwarp, warp, lane);
    int kbest = -1, phase = -1, phibest = -1;
    if (key != FS_KEY_NONE) {
      const float band = __fmul_rn(1.02f, fs_unorderable((uint32_t)key));
      key = FS_KEY_NONE;                                 // (most memory, largest SM_free, lowest k)
      for (int k = tid; k < v.K; k += nthr) {
        const fs_gpu_avail w = work[k];
        const CmEval e = cm_eval(v, c, k, w, -1);
        if (e.ok && e.ev.e <= band) {
          const unsigned long long kk = ((unsigned long long)(~fs_orderable(w.mem_free_mb)) << 32) |
                                        ((unsigned long long)(uint32_t)(d.S - e.p.smf) << 24) | (uint32_t)k;
          key = kk < key ? kk : key;
        }
      }
      key = cm_block_min(key, s_buf, par, nwarp, warp, lane);
      kbest = (int)((uint32_t)key & 0xFFFFFFu); phase = 1;
    } else {
      // ---- Phase 3: F_max retry, first feasible GPU in T_avail order ----------------------------
      for (int k = tid; k < v.K; k += nthr) {
        const fs_gpu_avail w = work[k];
        const CmEval e = cm_eval(v, c, k, w, d.F - 1);
        if (e.ok) {
          const unsigned long long kk = ((unsigned long long)fs_orderable(w.t_avail_ms) << 32) | (uint32_t)k;
          key = kk < key ? kk : key;
        }
      }
      key = cm_block_min(key, s_buf, par, nwarp, warp, lane);
      if (key != FS_KEY_NONE) { kbest = (int)(uint32_t)key; phase = 2; phibest = d.F - 1; }
    }
    if (kbest >= 0) {
      if (tid == kbest % nthr) {                         // the owner writes the decision and commits it
        fs_gpu_avail w = work[kbest];
        if (phase == 1) phibest = w.f_cur;
        const CmEval e = cm_eval(v, c, kbest, w, phibest);
        o.gpu = kbest; o.sigma = (int16_t)(e.p.smf - 1); o.phi = (int16_t)phibest; o.beta = (int16_t)e.p.br1;
        o.f_req = (int16_t)phase; o.energy_mj = e.ev.e; o.ttft_ms = e.ev.ttft; o.tbt_ms = e.ev.tbt;
        o.flat = (uint32_t)((kbest * d.S + e.p.smf - 1) * d.F + phibest);
        out[r] = o;
        const float tdec = c.O > 0 ? __fmul_rn(__uint2float_rn(e.p.rounds1), e.ev.tbt) : 0.f;
        w.t_avail_ms = __fadd_rn(e.ev.ttft, tdec);
        w.mem_free_mb = __fsub_rn(w.mem_free_mb, c.mem);
        w.f_cur = phibest;
        work[kbest] = w;
      }
    } else if (warp == 0) {
      // ---- scale-out: energy-optimal feasible frequency of a fresh GPU; no record changes -------
      key = FS_KEY_NONE;
      for (int phi = lane; phi < d.F; phi += 32) {
        const OwnEval ev = own_eval_planes(v, c, 0, c.O, c.load_ms, d.S - 1, phi);
        if (ev.ok) { const unsigned long long kk = fs_make_key(ev.e, (uint32_t)phi); key = kk < key ? kk : key; }
      }
      key = fs_warp_min_key(key);
      if (key != FS_KEY_NONE) {
        const int phi = (int)(uint32_t)key;
        const OwnEval ev = own_eval_planes(v, c, 0, c.O, c.load_ms, d.S - 1, phi);
        o.sigma = (int16_t)(d.S - 1); o.phi = (int16_t)phi; o.beta = 0; o.f_req = 3;
        o.energy_mj = ev.e; o.ttft_ms = ev.ttft; o.tbt_ms = ev.tbt;
      }
      if (lane == 0) out[r] = o;
    }
  }
}

// The same pass with the GPUs in registers: thread t keeps the records of GPUs t, t + blockDim, ...
// (KPT of them), so K <= KPT * blockDim.  The table entries of request r+1 at each GPU's F_curr are
// requested right after request r has been scored and arrive while r's two reductions and its commit
// run; a GPU whose F_curr the commit changed reloads its four entries.  What remains on the serial chain
// of a request is arithmetic and two block-wide minima.
// ---- thread-block cluster helpers (sm_90+ PTX): rank, size, a peer block's shared memory, barrier ----
__device__ __forceinline__ uint32_t cl_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cl_size() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cl_store_u64(const void* local_smem, uint32_t peer, unsigned long long x) {
  uint32_t remote;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(fs_smem_u32(local_smem)), "r"(peer));
  asm volatile("st.shared::cluster.u64 [%0], %1;" ::"r"(remote), "l"(x) : "memory");
}
__device__ __forceinline__ void cl_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
constexpr int CM_MAXC = 8;                        // portable cluster size

// minimum over the block and, with CLUSTER, over the blocks of the cluster: every block's leader warp
// stores the block's minimum into slot [par][own rank] of every block (distributed shared memory), one
// cluster barrier, every thread reads the slots of its own block
template <bool CLUSTER>
__device__ __forceinline__ unsigned long long cm_min_all(unsigned long long x, unsigned long long (*buf)[CM_THREADS / 32],
                                                         unsigned long long (*cbuf)[CM_MAXC], int& par, int nwarp,
                                                         int warp, int lane, uint32_t crank, uint32_t csize) {
  if (!CLUSTER) return cm_block_min(x, buf, par, nwarp, warp, lane);
  const int p = par;
  x = cm_block_min(x, buf, par, nwarp, warp, lane);
  if (warp == 0 && lane < (int)csize) cl_store_u64(&cbuf[p][crank], (uint32_t)lane, x);
  cl_sync();
  unsigned long long y = lane < (int)csize ? cbuf[p][lane] : FS_KEY_NONE;
  return fs_warp_min_key(y);
}

struct CmPre { float l0, p0, l1, p1; int phi; };

__device__ __forceinline__ CmPre cm_preload(const FsView& v, const ReqCtx& c, const FsGpuInfo& gi) {
  CmPre q; q.l0 = q.p0 = q.l1 = q.p1 = 1.f; q.phi = -1;
  if (!c.valid || gi.n_res < 1 || gi.sm_free < 1) return q;
  const PairCtx p = make_pair(v, c, gi);                 // br1 depends on the tenants only
  const FsDimsDev& d = v.d;
  const size_t o = (size_t)(gi.sm_free - 1) * d.F + gi.f_cur;
  const size_t i0 = fs_plane(d, c.m, 0, c.br0) + o, i1 = fs_plane(d, c.m, 1, p.br1) + o;
  const float2 a = v.lpT[i0], b = v.lpT[i1];
  q.l0 = a.x; q.p0 = a.y; q.l1 = b.x; q.p1 = b.y; q.phi = gi.f_cur;
  return q;
}

constexpr int CMR_THREADS = 512;                  // 128 registers per thread: the records of up to 4 GPUs
template <int KPT, bool CLUSTER>
__global__ void __launch_bounds__(CMR_THREADS) dispatch_commit_reg_kernel(FsView v, int R,
                                                                         const fs_request* __restrict__ reqs,
                                                                         fs_placement* __restrict__ out,
                                                                         fs_gpu_avail* __restrict__ work) {
  __shared__ unsigned long long s_buf[2][CM_THREADS / 32];
  __shared__ unsigned long long s_cbuf[2][CM_MAXC];
  const FsDimsDev d = v.d;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const uint32_t crank = CLUSTER ? cl_rank() : 0u, csize = CLUSTER ? cl_size() : 1u;
  // thread `tid` of `nthr` across the cluster owns GPUs tid, tid + nthr, ...
  const int tid = (int)crank * (int)blockDim.x + (int)threadIdx.x, nthr = (int)csize * (int)blockDim.x;
  int par = 0;
  FsGpuInfo gi[KPT]; CmPre pre[KPT];
#pragma unroll
  for (int u = 0; u < KPT; ++u) {
    const int k = tid + u * nthr;
    if (k < v.K) gi[u] = v.ginfo[k];
    else { gi[u] = FsGpuInfo{}; gi[u].n_res = 0; }
  }
  fs_request rq_nx{};                                  // the raw request after the next one to be scored
  if (R > 0) rq_nx = reqs[0];
  ReqCtx cn = make_req(v, rq_nx);
  if (R == 0) cn.valid = false;
  if (R > 1) rq_nx = reqs[1];
#pragma unroll
  for (int u = 0; u < KPT; ++u) pre[u] = cm_preload(v, cn, gi[u]);
  for (int r = 0; r < R; ++r) {
    fs_placement o;
    o.gpu = -1; o.sigma = o.phi = o.beta = o.f_req = -1;
    o.energy_mj = o.ttft_ms = o.tbt_ms = FS_INF; o.flat = 0xFFFFFFFFu; o._pad = 0;
    const ReqCtx c = cn;
    // ---- score request r at F_curr from the entries requested one request ago --------------------
    float ce[KPT], cttft[KPT], ctbt[KPT]; bool cok[KPT];
    unsigned long long key = FS_KEY_NONE;
#pragma unroll
    for (int u = 0; u < KPT; ++u) {
      cok[u] = false; ce[u] = FS_INF; cttft[u] = FS_INF; ctbt[u] = FS_INF;
      if (!c.valid) continue;
      const PairCtx p = make_pair(v, c, gi[u]);
      if (!p.ok) continue;
      if (pre[u].phi != gi[u].f_cur) pre[u] = cm_preload(v, c, gi[u]);   // the last commit moved this GPU's clock
      const OwnEval ev = own_eval_vals(c, p.rounds1, p.wait, pre[u].l0, pre[u].p0, pre[u].l1, pre[u].p1);
      cok[u] = ev.ok; ce[u] = ev.e; cttft[u] = ev.ttft; ctbt[u] = ev.tbt;
      if (ev.ok) { const unsigned long long kk = fs_orderable(ev.e); key = kk < key ? kk : key; }
    }
    // ---- request r+1: its context, and its table entries on the way -------------------------------
    if (r + 1 < R) {
      cn = make_req(v, rq_nx);
      if (r + 2 < R) rq_nx = reqs[r + 2];
#pragma unroll
      for (int u = 0; u < KPT; ++u) pre[u] = cm_preload(v, cn, gi[u]);
    }
    if (!c.valid) { if (tid == 0) { fs_raise(v.flag, FS_FLAG_REQUEST); out[r] = o; } continue; }
    key = cm_min_all<CLUSTER>(key, s_buf, s_cbuf, par, nwarp, warp, lane, crank, csize);
    int kbest = -1, phase = -1;
    if (key != FS_KEY_NONE) {
      const float band = __fmul_rn(1.02f, fs_unorderable((uint32_t)key));
      key = FS_KEY_NONE;                                 // (most memory, largest SM_free, lowest k)
#pragma unroll
      for (int u = 0; u < KPT; ++u)
        if (cok[u] && ce[u] <= band) {
          const unsigned long long kk = ((unsigned long long)(~fs_orderable(gi[u].mem_free_mb)) << 32) |
                                        ((unsigned long long)(uint32_t)(d.S - gi[u].sm_free) << 24) | (uint32_t)(tid + u * nthr);
          key = kk < key ? kk : key;
        }
      key = cm_min_all<CLUSTER>(key, s_buf, s_cbuf, par, nwarp, warp, lane, crank, csize);
      kbest = (int)((uint32_t)key & 0xFFFFFFu); phase = 1;
    } else {
      // ---- Phase 3: F_max retry, first feasible GPU in T_avail order ----------------------------
#pragma unroll
      for (int u = 0; u < KPT; ++u) {
        cok[u] = false;
        const PairCtx p = make_pair(v, c, gi[u]);
        if (!p.ok) continue;
        const OwnEval ev = own_eval_planes(v, c, p.br1, p.rounds1, p.wait, p.smf - 1, d.F - 1);
        cok[u] = ev.ok; ce[u] = ev.e; cttft[u] = ev.ttft; ctbt[u] = ev.tbt;
        if (ev.ok) {
          const unsigned long long kk = ((unsigned long long)fs_orderable(gi[u].t_avail_ms) << 32) | (uint32_t)(tid + u * nthr);
          key = kk < key ? kk : key;
        }
      }
      key = cm_min_all<CLUSTER>(key, s_buf, s_cbuf, par, nwarp, warp, lane, crank, csize);
      if (key != FS_KEY_NONE) { kbest = (int)(uint32_t)key; phase = 2; }
    }
    if (kbest >= 0) {
#pragma unroll
      for (int u = 0; u < KPT; ++u)
        if (kbest == tid + u * nthr) {                   // the owner writes the decision and commits it
          const PairCtx p = make_pair(v, c, gi[u]);
          const int phibest = phase == 1 ? gi[u].f_cur : d.F - 1;
          o.gpu = kbest; o.sigma = (int16_t)(p.smf - 1); o.phi = (int16_t)phibest; o.beta = (int16_t)p.br1;
          o.f_req = (int16_t)phase; o.energy_mj = ce[u]; o.ttft_ms = cttft[u]; o.tbt_ms = ctbt[u];
          o.flat = (uint32_t)((kbest * d.S + p.smf - 1) * d.F + phibest);
          out[r] = o;
          const float tdec = c.O > 0 ? __fmul_rn(__uint2float_rn(p.rounds1), ctbt[u]) : 0.f;
          gi[u].t_avail_ms = __fadd_rn(cttft[u], tdec);
          gi[u].mem_free_mb = __fsub_rn(gi[u].mem_free_mb, c.mem);
          gi[u].f_cur = phibest;
        }
    } else if (warp == 0 && crank == 0) {
      // ---- scale-out: energy-optimal feasible frequency of a fresh GPU; no record changes -------
      key = FS_KEY_NONE;
      for (int phi = lane; phi < d.F; phi += 32) {
        const OwnEval ev = own_eval_planes(v, c, 0, c.O, c.load_ms, d.S - 1, phi);
        if (ev.ok) { const unsigned long long kk = fs_make_key(ev.e, (uint32_t)phi); key = kk < key ? kk : key; }
      }
      key = fs_warp_min_key(key);
      if (key != FS_KEY_NONE) {
        const int phi = (int)(uint32_t)key;
        const OwnEval ev = own_eval_planes(v, c, 0, c.O, c.load_ms, d.S - 1, phi);
        o.sigma = (int16_t)(d.S - 1); o.phi = (int16_t)phi; o.beta = 0; o.f_req = 3;
        o.energy_mj = ev.e; o.ttft_ms = ev.ttft; o.tbt_ms = ev.tbt;
      }
      if (lane == 0) out[r] = o;
    }
  }
  if (CLUSTER) cl_sync();                              // no block leaves while a peer may still store into it
#pragma unroll
  for (int u = 0; u < KPT; ++u) {
    const int k = tid + u * nthr;
    if (k < v.K) {
      fs_gpu_avail w; w.t_avail_ms = gi[u].t_avail_ms; w.mem_free_mb = gi[u].mem_free_mb; w.f_cur = gi[u].f_cur; w._pad = 0;
      work[k] = w;
    }
  }
}

}  // namespace

int fsk_place_smem_attr() {
  int e = 0;
#define FS_ATTR_DENSE(NP, VC, CL) \
  e |= (int)cudaFuncSetAttribute(place_dense_kernel<NP, VC, CL>, cudaFuncAttributeMaxDynamicSharedMemorySize, DENSE_SMEM_MAX)
  FS_ATTR_DENSE(1, false, false); FS_ATTR_DENSE(2, false, false); FS_ATTR_DENSE(2, true, false);
  FS_ATTR_DENSE(2, false, true);  FS_ATTR_DENSE(2, true, true);
#undef FS_ATTR_DENSE
  e |= (int)cudaFuncSetAttribute(dispatch_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DISP_WARPS * 2 * FS_MAX_S * 32 * 4);
  e |= (int)cudaFuncSetAttribute(dispatch_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DISP_WARPS * 2 * FS_MAX_S * 64 * 4);
  return e;
}

int fsk_place(const FsView& v, int R, const fs_request* reqs, fs_placement* out,
              const FsPlaceScratch& sc, cudaStream_t st, FsTimers* tm) {
  if (R <= 0) return 0;
  int launches = 0;
  if (sc.count_work) cudaMemsetAsync(sc.stats, 0, sizeof(unsigned long long) * FS_NSTATS, st);
  if (v.K <= 0) {
    cudaMemsetAsync(sc.keys, 0xFF, sizeof(unsigned long long) * (size_t)R, st);
    place_decode_kernel<<<(R + 7) / 8, 256, 0, st>>>(v, R, reqs, sc.keys, out);
    return 1;
  }
  fs_tm_beg(tm, FS_T_PLACE_SCORE, st);
  // one persistent block per SM.  Warps per block: as many as fit (shared memory: one tile per warp;
  // registers cap them at DENSE_MAXW), fewer when R alone cannot occupy every SM.
  const int FT = v.d.F <= 32 ? 32 : 64;
  const int ncb = (v.d.F + 63) / 64;                 // column blocks of 64 frequencies (1 unless F > 64)
  const int nchunk = v.Kpad / FS_CHUNK;
  const size_t pw = dense_warp_bytes(v.d.S, FT);
  int W = (int)(DENSE_SMEM_MAX / pw);
  W = max(1, min(min(DENSE_MAXW, W), (R + sc.sm_count - 1) / sc.sm_count));
  // the GPUs are cut into slices only when the requests alone cannot occupy every SM
  int nslice = 1;
  const int nbatch = (R + W - 1) / W;
  if (nbatch * ncb < sc.sm_count) nslice = min(nchunk, (sc.sm_count + nbatch * ncb - 1) / (nbatch * ncb));
  const int cps = (nchunk + nslice - 1) / nslice;
  nslice = (nchunk + cps - 1) / cps;
  const int nsc = nslice * ncb;
  const int streams = max(1, min(nbatch, sc.sm_count / nsc));
  const int grid = streams * nsc;
  const size_t smem = dense_smem_bytes(W, v.d.S, FT);
  cudaMemsetAsync(sc.ctr, 0, sizeof(unsigned int) * (size_t)nsc, st);
  // one slice: the scoring kernel writes the placement records itself (no key array, no decode launch)
  fs_placement* direct = nsc == 1 ? out : nullptr;
  if (!direct) cudaMemsetAsync(sc.keys, 0xFF, sizeof(unsigned long long) * (size_t)R, st);
  unsigned long long* stats = sc.count_work ? sc.stats : nullptr;
#define FS_LAUNCH_DENSE(NP, VC, CL) \
  place_dense_kernel<NP, VC, CL><<<grid, W * 32, smem, st>>>(v, R, reqs, sc.keys, nslice, ncb, cps, sc.ctr, sc.warm_off, sc.witems, stats, direct)
  const bool vec = FT == 64 && (v.d.F & 1) == 0;
  if (FT == 32) FS_LAUNCH_DENSE(1, false, false);
  else if (ncb == 1) { if (vec) FS_LAUNCH_DENSE(2, true, false); else FS_LAUNCH_DENSE(2, false, false); }
  else               { if (vec) FS_LAUNCH_DENSE(2, true, true);  else FS_LAUNCH_DENSE(2, false, true); }
#undef FS_LAUNCH_DENSE
  ++launches;
  fs_tm_end(tm, FS_T_PLACE_SCORE, st);
  if (direct) return launches;
  fs_tm_beg(tm, FS_T_PLACE_DECODE, st);
  place_decode_kernel<<<(R + 7) / 8, 256, 0, st>>>(v, R, reqs, sc.keys, out);
  fs_tm_end(tm, FS_T_PLACE_DECODE, st);
  ++launches;
  return launches;
}

int fsk_dispatch(const FsView& v, int R, const fs_request* reqs, fs_placement* out, const int32_t* warm_off,
                 const FsWarmItem* witems, cudaStream_t st, FsTimers* tm) {
  if (R <= 0) return 0;
  const int use_tiles = v.d.F <= 64;
  const int FT = v.d.F <= 32 ? 32 : 64;
  // few requests: one block per request, its warps split the GPUs; batches: one warp per request
  const bool block_mode = (long long)R * DISP_WARPS <= 2LL * 148 * DISP_WARPS && v.Kpad >= 64 * DISP_WARPS;
  const size_t smem = use_tiles ? (size_t)(block_mode ? 1 : DISP_WARPS) * 2 * v.d.S * FT * sizeof(float) : 0;
  fs_tm_beg(tm, FS_T_DISPATCH, st);
  const int grid = block_mode ? R : (R + DISP_WARPS - 1) / DISP_WARPS;
  if (FT == 32) {
    if (block_mode) dispatch_kernel<1, true><<<grid, DISP_WARPS * 32, smem, st>>>(v, R, reqs, out, use_tiles, warm_off, witems);
    else            dispatch_kernel<1, false><<<grid, DISP_WARPS * 32, smem, st>>>(v, R, reqs, out, use_tiles, warm_off, witems);
  } else {
    if (block_mode) dispatch_kernel<2, true><<<grid, DISP_WARPS * 32, smem, st>>>(v, R, reqs, out, use_tiles, warm_off, witems);
    else            dispatch_kernel<2, false><<<grid, DISP_WARPS * 32, smem, st>>>(v, R, reqs, out, use_tiles, warm_off, witems);
  }
  fs_tm_end(tm, FS_T_DISPATCH, st);
  return 1;
}

int fsk_dispatch_commit(const FsView& v, int R, const fs_request* reqs, fs_placement* out, fs_gpu_avail* work,
                        cudaStream_t st, FsTimers* tm) {
  if (R <= 0 && v.K <= 0) return 0;
  int threads = ((v.K + 31) / 32) * 32;
  threads = threads < 32 ? 32 : (threads > CM_THREADS ? CM_THREADS : threads);
  fs_tm_beg(tm, FS_T_DISPATCH, st);
  const int tr = threads > CMR_THREADS ? CMR_THREADS : threads;
  if (v.K <= CMR_THREADS) dispatch_commit_reg_kernel<1, false><<<1, tr, 0, st>>>(v, R, reqs, out, work);
  else if (v.K <= 2 * CMR_THREADS) dispatch_commit_reg_kernel<2, false><<<1, tr, 0, st>>>(v, R, reqs, out, work);
  else if (v.K <= 4 * CMR_THREADS) dispatch_commit_reg_kernel<4, false><<<1, tr, 0, st>>>(v, R, reqs, out, work);
  else if (v.K <= CM_MAXC * 4 * CMR_THREADS) {
    // a thread-block cluster: up to 8 blocks x 512 threads x 4 GPUs in registers, minima through
    // distributed shared memory
    const int csize = (v.K + 4 * CMR_THREADS - 1) / (4 * CMR_THREADS);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)csize); cfg.blockDim = dim3(CMR_THREADS); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)csize; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, dispatch_commit_reg_kernel<4, true>, v, R, reqs, out, work);
  }
  else dispatch_commit_kernel<<<1, threads, 0, st>>>(v, R, reqs, out, work);
  fs_tm_end(tm, FS_T_DISPATCH, st);
  return 1;
}
