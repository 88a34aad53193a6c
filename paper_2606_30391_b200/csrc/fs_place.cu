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

int fsk_place(const FsView& v, int R, const fs_request* reqs, fs_placement* out,
              const FsPlaceScratch& sc, cudaStream_t st, FsTimers* tm) {
  if (R <= 0) return 0;
  int launches = 0;
  cudaMemsetAsync(sc.keys, 0xFF, sizeof(unsigned long long) * (size_t)R, st);
  cudaMemsetAsync(sc.stats, 0, sizeof(unsigned long long) * 2, st);
  if (v.K <= 0) {
    place_decode_kernel<<<(R + 7) / 8, 256, 0, st>>>(v, R, reqs, sc.keys, out);
    return 1;
  }
  // split the GPUs of one request over several warps when R alone cannot fill 148 SMs
  const long long want_warps = 148LL * 32;
  int nsplit = 1;
  if (R < want_warps) nsplit = (int)((want_warps + R - 1) / R);
  if (nsplit > v.K) nsplit = v.K > 0 ? v.K : 1;
  const int kchunk = (v.K + nsplit - 1) / nsplit;
  nsplit = (v.K + kchunk - 1) / (kchunk > 0 ? kchunk : 1);
  if (nsplit < 1) nsplit = 1;
  const long long warps = (long long)R * nsplit;
  fs_tm_beg(tm, FS_T_PLACE_SCORE, st);
  place_generic_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(v, R, reqs, sc.keys, nsplit,
                                                                   kchunk, sc.stats);
  fs_tm_end(tm, FS_T_PLACE_SCORE, st);
  ++launches;
  fs_tm_beg(tm, FS_T_PLACE_DECODE, st);
  place_decode_kernel<<<(R + 7) / 8, 256, 0, st>>>(v, R, reqs, sc.keys, out);
  fs_tm_end(tm, FS_T_PLACE_DECODE, st);
  ++launches;
  return launches;
}
