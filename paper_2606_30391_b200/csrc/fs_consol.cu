// fs_consol.cu — fs_consolidate: drain-one-source scoring over all GPU pairs (§3.5,
// R:s17-s20).  Per tenant and frequency the minimum feasible share (P:252 rule (1));
// 5 % safety margin on SMs and memory; idle power vs migration energy.
//
//   need_g[phi] = sum_i (sigma_i(phi)+1),  E_g[phi] = slot-order sum of e_i at those shares
//   C*_g   = min_phi { E_g[phi] : need_g[phi] <= S_eff }
//   C*_ab  = min_phi { fl(E_b[phi]+E_a[phi]) : need_a[phi]+need_b[phi] <= S_eff }  (lowest phi)
//   score(a->b) = fl(C*_ab - C*_b);   dst(a) = argmin_b (score, b)  as one 64-bit key
#include <cuda_fp16.h>

#include "fs_kernels.h"

namespace {

constexpr int TA = 8;          // sources per block of the pair kernel
constexpr int PAIR_THREADS = 256;

// ---- a9: per GPU, lanes over phi ------------------------------------------------------------
__global__ void __launch_bounds__(128) consol_agg_kernel(FsView v, int S_eff,
                                                        uint8_t* __restrict__ need,
                                                        float* __restrict__ E,
                                                        float4* __restrict__ agg) {
  const int lane = threadIdx.x & 31;
  const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (g >= v.K) return;
  const FsDimsDev d = v.d;
  const int n = v.ginfo[g].n_res;
  const fs_gpu_state& st = v.states[g];
  unsigned long long key = FS_KEY_NONE;
  // per tenant, independent of (phi, sigma): plane offsets, round counts (the divisions once), deadlines
  size_t o0[FS_RMAX], o1[FS_RMAX]; float r0[FS_RMAX], r1[FS_RMAX], slo0[FS_RMAX], slo1[FS_RMAX];
  bool has0[FS_RMAX], has1[FS_RMAX];
#pragma unroll
  for (int i = 0; i < FS_RMAX; ++i) {
    o0[i] = o1[i] = 0; r0[i] = r1[i] = 0.f; slo0[i] = slo1[i] = 0.f; has0[i] = has1[i] = false;
    if (i < n) {
      const fs_tenant& t = st.t[i];
      has0[i] = t.q[0] > 0; has1[i] = t.q[1] > 0; slo0[i] = t.slo_ms[0]; slo1[i] = t.slo_ms[1];
      o0[i] = fs_plane(d, t.model, 0, t.beta[0]); o1[i] = fs_plane(d, t.model, 1, t.beta[1]);
      r0[i] = __uint2float_rn(fs_ceil_div(t.q[0], t.beta[0] + 1u));
      r1[i] = __uint2float_rn(fs_ceil_div(t.q[1], t.beta[1] + 1u));
    }
  }
  for (int phi = lane; phi < d.F; phi += 32) {
    int nd = 0; float e = 0.0f; bool all = n >= 1;
#pragma unroll
    for (int i = 0; i < FS_RMAX; ++i) {
      if (i < n && all) {
        // lowest feasible share of tenant i at phi: four shares' table entries are requested together
        // (one memory latency per four shares instead of one per share), then tested in order
        int smin = -1; float ei = FS_INF;
        for (int sg0 = 0; sg0 < d.S && smin < 0; sg0 += 4) {
          float l0[4], p0[4], l1[4], p1[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const size_t o = (size_t)min(sg0 + u, d.S - 1) * d.F + phi;
            const float2 e0 = v.lpT[o0[i] + o], e1 = v.lpT[o1[i] + o];
            l0[u] = e0.x; p0[u] = e0.y; l1[u] = e1.x; p1[u] = e1.y;
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (smin < 0 && sg0 + u < d.S) {
              bool ok = true; float e0 = 0.0f, e1 = 0.0f;
              if (has0[i]) { const FsSlot sl = fs_slot_f(0, l0[u], p0[u], r0[i], 0.0f, slo0[i]); ok = sl.ok; e0 = sl.e; }
              if (has1[i]) { const FsSlot sl = fs_slot_f(1, l1[u], p1[u], r1[i], 0.0f, slo1[i]); ok = ok && sl.ok; e1 = sl.e; }
              if (ok) { smin = sg0 + u; ei = __fadd_rn(e0, e1); }
            }
          }
        }
        if (smin < 0) all = false;
        else { nd += smin + 1; e = (i == 0) ? ei : __fadd_rn(e, ei); }
      }
    }
    need[(size_t)phi * v.K + g] = all ? (uint8_t)nd : (uint8_t)FS_NEED_INF;
    E[(size_t)phi * v.K + g] = all ? e : FS_INF;
    if (all && nd <= S_eff && e < FS_INF) {
      const unsigned long long kk = fs_make_key(e, (uint32_t)phi);
      key = kk < key ? kk : key;
    }
  }
  key = fs_warp_min_key(key);
  if (lane == 0) {
    float mem = 0.0f, mig = 0.0f;
    for (int i = 0; i < n; ++i) {
      mem = (i == 0) ? st.t[i].mem_used_mb : __fadd_rn(mem, st.t[i].mem_used_mb);
      const float mg = v.models[st.t[i].model].mig_mj;
      mig = (i == 0) ? mg : __fadd_rn(mig, mg);
    }
    const float cstar = key == FS_KEY_NONE ? FS_INF : fs_unorderable((uint32_t)(key >> 32));
    agg[g] = make_float4(mem, cstar, mig, __int_as_float(n));
  }
}

// ---- what the pair kernel streams per destination: per frequency PAIR one {E[phi], E[phi+1]} and one packed
// pair of binary16 values S_eff - need (small integers: exact); a frequency past F-1 is never feasible.
// One more row than ceil(F/2) is allocated: the pair kernel's prefetch of the trip after the last needs no clamp.
__global__ void consol_pack_kernel(int K, int F, int S_eff, const uint8_t* __restrict__ need, const float* __restrict__ E,
                                   float2* __restrict__ E2, uint32_t* __restrict__ T2) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x, pp = blockIdx.y;
  if (b >= K) return;
  const int p0 = 2 * pp, p1 = 2 * pp + 1;
  const bool h1 = p1 < F;
  const float e1 = h1 ? E[(size_t)p1 * K + b] : FS_INF;
  const int n0 = (int)need[(size_t)p0 * K + b], n1 = h1 ? (int)need[(size_t)p1 * K + b] : FS_NEED_INF;
  const __half2 t = __halves2half2(__int2half_rn(S_eff - n0), __int2half_rn(S_eff - n1));
  E2[(size_t)pp * K + b] = make_float2(E[(size_t)p0 * K + b], e1);
  T2[(size_t)pp * K + b] = *reinterpret_cast<const uint32_t*>(&t);
}

// ---- a10: pair scoring; one block = TA sources x all destinations ----------------------------
__global__ void __launch_bounds__(PAIR_THREADS) consol_pair_kernel(
    FsView v, int S_eff, float mem_cap_mb, int delta_pct, const uint8_t* __restrict__ need, const float* __restrict__ E,
    const float2* __restrict__ E2, const uint32_t* __restrict__ T2,
    const float4* __restrict__ agg, unsigned long long* __restrict__ keys) {
  extern __shared__ unsigned char smem_raw[];
  // M_eff = fl(fl(cap * (100 - delta)) / 100): the 5 % margin on memory (R:s19)
  const float M_eff = __fdiv_rn(__fmul_rn(mem_cap_mb, (float)(100 - delta_pct)), 100.0f);
  const int F = v.d.F, K = v.K;
  // [ceil(F/2)][TA] {E_a[phi], E_a[phi+1], need_a of both as two binary16 values, -}: one LDS.128 per source and
  // frequency pair, read by broadcast; a frequency past F-1 is never feasible (E = INF, need = FS_NEED_INF)
  float4* sEN = reinterpret_cast<float4*>(smem_raw);
  __shared__ unsigned long long sred[TA][PAIR_THREADS / 32];
  const int a0 = blockIdx.x * TA, FP = (F + 1) / 2;
  for (int x = threadIdx.x; x < FP * TA; x += blockDim.x) {
    const int pp = x / TA, a = a0 + x % TA, p0 = 2 * pp, p1 = 2 * pp + 1;
    const bool h0 = a < K, h1 = a < K && p1 < F;
    const float e0 = h0 ? E[(size_t)p0 * K + a] : FS_INF, e1 = h1 ? E[(size_t)p1 * K + a] : FS_INF;
    const int n0 = h0 ? (int)need[(size_t)p0 * K + a] : FS_NEED_INF, n1 = h1 ? (int)need[(size_t)p1 * K + a] : FS_NEED_INF;
    const __half2 nn = __halves2half2(__int2half_rn(n0), __int2half_rn(n1));     // small integers: exact
    sEN[x] = make_float4(e0, e1, __uint_as_float(*reinterpret_cast<const uint32_t*>(&nn)), 0.0f);
  }
  __syncthreads();
  float4 ag[TA];
#pragma unroll
  for (int t = 0; t < TA; ++t) ag[t] = a0 + t < K ? agg[a0 + t] : make_float4(0.f, FS_INF, 0.f, 0.f);
  unsigned long long best[TA];
#pragma unroll
  for (int t = 0; t < TA; ++t) best[t] = FS_KEY_NONE;
  // two destinations per thread and trip: the broadcast read of a source's (E, need) serves both; per
  // (source, destination, phi) one add, one integer compare and one predicated min
  // blockIdx.y = a slice of the destinations (finer blocks: the grid is several waves deep and its tail short);
  // the slices' minima meet in keys[] by atomicMin
  const int per = (K + (int)gridDim.y - 1) / (int)gridDim.y;
  const int bs = blockIdx.y * per, be = min(K, bs + per);
  for (int b0 = bs + threadIdx.x; b0 < be; b0 += 2 * blockDim.x) {
    const int b1 = b0 + blockDim.x;
    const bool two = b1 < be;
    const int b1c = two ? b1 : b0;
    float cab0[TA], cab1[TA];
#pragma unroll
    for (int t = 0; t < TA; ++t) cab0[t] = cab1[t] = FS_INF;
    // two frequencies per trip, software-pipelined: the eight values of the NEXT trip (E and need of both
    // destinations) are requested before the current trip's 2 x TA x 2 candidates are scored, so the loads'
    // latency hides behind the arithmetic (the kernel waited on them for 40 % of its issue slots before)
    // Two frequencies per trip.  Per (source, destination, frequency pair): ONE packed binary16 compare gives both
    // feasibility predicates (need_a + need_b <= S_eff  <=>  need_a <= S_eff - need_b; HSETP2), two adds, two
    // selects of +INF and one three-input min (FMNMX3): 3.25 instructions per (pair, frequency) instead of 4, and
    // half the work of the ALU pipe, which bound this kernel.
    // The destinations' values come packed per frequency pair (consol_pack_kernel): one 64-bit and one 32-bit load
    // per destination and trip, on running pointers.  Software-pipelined: the next trip's values are requested
    // before this trip is scored (one row of padding behind the last pair: no clamp).
    float ec[2][2]; uint32_t tc[2];                      // E [phi in trip][destination]; S_eff - need of both phis, packed, [destination]
    const float2* pe0 = E2 + b0; const float2* pe1 = E2 + b1c;
    const uint32_t* pt0 = T2 + b0; const uint32_t* pt1 = T2 + b1c;
#define FS_PAIR_LOAD(EC, TC)                                                                              \
    {                                                                                                     \
      const float2 x0 = *pe0, x1 = *pe1;                                                                  \
      EC[0][0] = x0.x; EC[1][0] = x0.y; EC[0][1] = x1.x; EC[1][1] = x1.y; TC[0] = *pt0; TC[1] = *pt1;     \
    }
    FS_PAIR_LOAD(ec, tc)
    const float4* sp = sEN;
    for (int pp = 0; pp < FP; ++pp) {
      pe0 += K; pe1 += K; pt0 += K; pt1 += K;
      float en_[2][2]; uint32_t tn_[2];
      FS_PAIR_LOAD(en_, tn_)
#pragma unroll
      for (int t = 0; t < TA; ++t) {
        const float4 en = sp[t];
        const uint32_t na2 = __float_as_uint(en.z);
        asm("{.reg .pred p, q; .reg .f32 y0, y1;\n\t"
            "setp.le.f16x2 p|q, %3, %4;\n\t"
            "selp.f32 y0, %1, 0f7F800000, p;\n\t"
            "selp.f32 y1, %2, 0f7F800000, q;\n\t"
            "min.f32 %0, %0, y0, y1;}"
            : "+f"(cab0[t]) : "f"(__fadd_rn(ec[0][0], en.x)), "f"(__fadd_rn(ec[1][0], en.y)), "r"(na2), "r"(tc[0]));
        asm("{.reg .pred p, q; .reg .f32 y0, y1;\n\t"
            "setp.le.f16x2 p|q, %3, %4;\n\t"
            "selp.f32 y0, %1, 0f7F800000, p;\n\t"
            "selp.f32 y1, %2, 0f7F800000, q;\n\t"
            "min.f32 %0, %0, y0, y1;}"
            : "+f"(cab1[t]) : "f"(__fadd_rn(ec[0][1], en.x)), "f"(__fadd_rn(ec[1][1], en.y)), "r"(na2), "r"(tc[1]));
      }
      sp += TA;
#pragma unroll
      for (int u = 0; u < 2; ++u) { ec[u][0] = en_[u][0]; ec[u][1] = en_[u][1]; }
      tc[0] = tn_[0]; tc[1] = tn_[1];
    }
#undef FS_PAIR_LOAD
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      if (h == 1 && !two) break;
      const int b = h ? b1 : b0;
      const float4 gb = agg[b];
      const int n_b = __float_as_int(gb.w);
#pragma unroll
      for (int t = 0; t < TA; ++t) {
        const float cab = h ? cab1[t] : cab0[t];
        const int a = a0 + t, n_a = __float_as_int(ag[t].w);
        const bool ok = a < K && a != b && n_a >= 1 && n_b >= 1 && n_a + n_b <= FS_RMAX &&
                        (__fadd_rn(ag[t].x, gb.x) <= M_eff) && gb.y < FS_INF && cab < FS_INF;
        if (ok) {
          const unsigned long long kk = fs_make_key(__fsub_rn(cab, gb.y), (uint32_t)b);
          best[t] = kk < best[t] ? kk : best[t];
        }
      }
    }
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int t = 0; t < TA; ++t) {
    const unsigned long long kk = fs_warp_min_key(best[t]);
    if (lane == 0) sred[t][warp] = kk;
  }
  __syncthreads();
  if (threadIdx.x < TA && a0 + threadIdx.x < K) {
    unsigned long long kk = FS_KEY_NONE;
    for (int w = 0; w < PAIR_THREADS / 32; ++w) kk = sred[threadIdx.x][w] < kk ? sred[threadIdx.x][w] : kk;
    if (kk != FS_KEY_NONE) atomicMin(&keys[a0 + threadIdx.x], kk);
  }
}

// ---- decode: dst, the merged GPU's frequency, score and net saving ---------------------------
__global__ void consol_decode_kernel(FsView v, int S_eff, fs_params prm,
                                     const uint8_t* __restrict__ need, const float* __restrict__ E,
                                     const float4* __restrict__ agg,
                                     const unsigned long long* __restrict__ keys,
                                     fs_consol_out* __restrict__ out) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= v.K) return;
  fs_consol_out o; o.dst = -1; o.phi = -1; o.score_mj = FS_INF; o.saving_mj = -FS_INF;
  const unsigned long long key = keys[a];
  if (key != FS_KEY_NONE) {
    const int b = (int)(uint32_t)key;
    float cab = FS_INF; int phis = -1;
    for (int phi = 0; phi < v.d.F; ++phi) {
      if ((int)need[(size_t)phi * v.K + a] + (int)need[(size_t)phi * v.K + b] > S_eff) continue;
      const float e = __fadd_rn(E[(size_t)phi * v.K + b], E[(size_t)phi * v.K + a]);
      if (e < cab) { cab = e; phis = phi; }            // strict: lowest phi on ties
    }
    const float4 ga = agg[a];
    o.dst = b; o.phi = phis; o.score_mj = fs_unorderable((uint32_t)(key >> 32));
    // saved idle energy over the horizon + the source's own optimum - what the destination
    // pays extra - migration energy (R:s18)
    o.saving_mj = __fsub_rn(__fadd_rn(__fmul_rn(prm.p_idle_w, prm.horizon_ms), ga.y),
                            __fadd_rn(o.score_mj, ga.z));
  }
  out[a] = o;
}

}  // namespace

int fsk_consolidate(const FsView& v, const fs_params& prm, fs_consol_out* out,
                    const FsConsolScratch& sc, cudaStream_t st, FsTimers* tm) {
  if (v.K <= 0) return 0;
  const int S_eff = (v.d.S * (100 - prm.delta_pct)) / 100;
  fs_tm_beg(tm, FS_T_CONSOL_AGG, st);
  consol_agg_kernel<<<(v.K + 3) / 4, 128, 0, st>>>(v, S_eff, sc.need, sc.E, sc.agg);
  fs_tm_end(tm, FS_T_CONSOL_AGG, st);
  const size_t smem = sizeof(float4) * ((v.d.F + 1) / 2) * TA;
  fs_tm_beg(tm, FS_T_CONSOL_PAIR, st);
  consol_pack_kernel<<<dim3((v.K + 255) / 256, (v.d.F + 1) / 2), 256, 0, st>>>(v.K, v.d.F, S_eff, sc.need, sc.E, sc.E2, sc.T2);
  cudaMemsetAsync(sc.keys, 0xFF, sizeof(unsigned long long) * (size_t)v.K, st);
  const int nds = max(1, min(8, v.K / (4 * PAIR_THREADS)));          // destination slices: >= 2 trips of 2 x 256 each
  consol_pair_kernel<<<dim3((v.K + TA - 1) / TA, nds), PAIR_THREADS, smem, st>>>(v, S_eff, prm.mem_cap_mb, prm.delta_pct,
                                                                    sc.need, sc.E, sc.E2, sc.T2, sc.agg, sc.keys);
  fs_tm_end(tm, FS_T_CONSOL_PAIR, st);
  consol_decode_kernel<<<(v.K + 127) / 128, 128, 0, st>>>(v, S_eff, prm, sc.need, sc.E, sc.agg,
                                                          sc.keys, out);
  return 4;
}
