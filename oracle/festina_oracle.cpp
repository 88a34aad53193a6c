// festina_oracle.cpp — TEST INFRASTRUCTURE, not the product.
//
// Plain, slow, obviously-correct CPU statement of what libfestina_eval computes, written from
// the paper text (arxiv/paper_2606_30391; "P:NNN" = line of PAPER.md) and the readings listed
// in DESIGN.md ("R:sNN").  Naive nested loops in the paper's order; no blocking, no hoisting,
// no shared code with the CUDA path (own struct definitions, own arithmetic).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// Each entry point returns an exact argmin over a finite candidate set under a fixed binary32
// evaluation order, so the oracle is that definition written out.  Pins (tests/, -m "not gpu"):
//   slot rule / energy .... Eq. 1-2 identity by hand, brute force
//   placement ............. Eq. 2-3 special case, brute-force enumeration with an
//                           independently written numpy evaluator, feasibility/optimality
//                           invariants, duplicate-GPU / duplicate-frequency tie cases,
//                           continuous optimum of the analytic generator
//   local config .......... Fig. 8 step 3 worked table, brute force
//   consolidation ......... brute force, C*_ab symmetry, empty-destination case,
//                           App. G arithmetic
//   paper dispatcher ...... Eq. 2-3 by hand, Fig. 6-shaped toy, 2 % band
//                           and tie-breaker cases, T_avail-ordered F_max retry and
//                           scale-out, independent numpy restatement
//   Alg. 1 phase 1 / EWR .. Eq. 8 and Little's law by hand, brute-force argmin restatement; EWR closed
//                           forms (0 iff aligned, two-LLM case by hand)
//   Alg. 1 phases 2-3 ..... BFD against brute-force optimal bin counts on tiny inputs (OPT <= BFD <=
//                           11/9 OPT + 1), a Fig. 9-shaped swap case by hand, capacity invariants
//   migration plan ........ brute force over all permutations (n <= 7), scipy's linear_sum_assignment,
//                           hand-built rule cases
//   priority batching ..... Fig. 8 steps 1-2 worked table, independent numpy
//                           restatement, budget / bypass invariants
// Nothing here is "parity unpinned".
//
// Build: g++ -O2 -ffp-contract=off -std=c++17 -shared -fPIC (see oracle/build.py).
// -ffp-contract=off matters: every fl(.) below is ONE binary32 rounding.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

constexpr int RMAX = 4;
const float INF = std::numeric_limits<float>::infinity();

struct Tenant {  // 28 B, layout of the state record
  int16_t model; uint8_t sigma, p0; uint8_t beta[2], p1[2];
  uint32_t q[2]; float slo_ms[2]; float mem_used_mb;
};
struct GpuState { int32_t n_res, f_cur; float t_avail_ms, mem_free_mb; Tenant t[RMAX]; };
struct Request { int32_t model; uint32_t L, o_pred; float slo_ttft_ms, slo_tbt_ms; uint32_t tag, pad[2]; };
struct ModelInfo { float load_ms, kv_mb_per_token, weights_mb, mig_mj; };
struct Placement { int32_t gpu; int16_t sigma, phi, beta, f_req; float energy_mj, ttft_ms, tbt_ms; uint32_t flat, pad; };
struct LocalCfg { int16_t phi, f_req; uint8_t sigma[RMAX]; uint8_t beta[RMAX][2]; float cost, energy_mj, power_w; uint32_t flat, pad[4]; };
struct ConsolOut { int32_t dst, phi; float score_mj, saving_mj; };
static_assert(sizeof(Tenant) == 28 && sizeof(GpuState) == 128 && sizeof(Request) == 32, "layout");
static_assert(sizeof(Placement) == 32 && sizeof(LocalCfg) == 48 && sizeof(ConsolOut) == 16, "layout");

struct Tables {  // LUT[model][phase][freq][SM share][batch] (axes R:s1)
  int M, F, S, B;
  const float* lat; const float* pow;
  size_t idx(int m, int p, int f, int s, int b) const {
    return ((((size_t)m * 2 + p) * F + f) * S + s) * B + b;
  }
  float LAT(int m, int p, int f, int s, int b) const { return lat[idx(m, p, f, s, b)]; }
  float POW(int m, int p, int f, int s, int b) const { return pow[idx(m, p, f, s, b)]; }
};

struct Slot { bool ok; float t, e; };

// Shared slot rule.  Energy = Power x Time (Eq. 1); deadline check at a frequency
// (P:216); "TBT for decode; TTFT for prefill" (R:s11):
//   rounds = ceil(q/(beta+1));  t = fl(rounds*LAT);  e = fl(t*POW)
//   prefill: fl(wait+t) <= slo     decode: LAT <= slo
Slot slot_eval(const Tables& T, int m, int p, int phi, int sigma, int beta, uint32_t q,
               float wait, float slo) {
  if (q == 0) return {true, 0.0f, 0.0f};
  uint32_t n = (uint32_t)beta + 1u;
  uint32_t rounds = (q + n - 1u) / n;
  float lat = T.LAT(m, p, phi, sigma, beta);
  float t = (float)rounds * lat;
  bool ok = (p == 0) ? ((wait + t) <= slo) : (lat <= slo);
  float e = t * T.POW(m, p, phi, sigma, beta);
  return {ok, t, e};
}

struct TenantEval { bool ok; float e; };

// One co-resident at frequency phi with its own share sigma_i, wait = 0 (its slo is already
// the remaining slack, R:s12).  bump = "one more sequence joins this tenant's decode batch":
// the decode bucket moves to beta+1 when the decode queue is non-empty; past the table => not ok.
TenantEval tenant_eval(const Tables& T, const Tenant& t, int phi, int sigma, bool bump) {
  int b1 = t.beta[1] + ((bump && t.q[1] > 0) ? 1 : 0);
  if (b1 >= T.B) return {false, INF};
  Slot s0 = slot_eval(T, t.model, 0, phi, sigma, t.beta[0], t.q[0], 0.0f, t.slo_ms[0]);
  Slot s1 = slot_eval(T, t.model, 1, phi, sigma, b1, t.q[1], 0.0f, t.slo_ms[1]);
  return {s0.ok && s1.ok, s0.e + s1.e};
}

int sm_free_of(const GpuState& g, int S) {
  int used = 0;
  for (int i = 0; i < g.n_res; ++i) used += g.t[i].sigma + 1;
  return S - used;
}

// ------------------------------------------------------------------------------------------
// fs_place_batch: global dispatch.  Phase 1 feasibility, Phase 2
// energy argmin (Eq. 2-3) generalised to (GPU, grant sigma, frequency phi)
// (R:s2-s5); F_max retry is inside the swept phi set.  Tie: lowest flat (R:s6).
void place_one(const Tables& T, const ModelInfo* mi, const GpuState* gs, int K,
               const Request& rq, Placement& out) {
  const int m = rq.model;
  const uint32_t O = (21u * rq.o_pred + 19u) / 20u;        // ceil(1.05*o_pred), R:s14
  const float mem = (float)(rq.L + O) * mi[m].kv_mb_per_token;  // Req_mem, R:s13
  bool have = false;
  float bestE = INF; uint32_t bestFlat = 0xFFFFFFFFu;
  Placement best{}; best.gpu = -1; best.sigma = best.phi = best.beta = best.f_req = -1;
  best.energy_mj = INF; best.ttft_ms = INF; best.tbt_ms = INF; best.flat = 0xFFFFFFFFu;

  for (int k = 0; k < K; ++k) {
    const GpuState& g = gs[k];
    if (g.n_res < 1) continue;                             // inactive GPU (R:s16)
    if (!(mem <= g.mem_free_mb)) continue;                 // memory must fit (R:s12)
    const int smf = sm_free_of(g, T.S);
    if (smf < 1) continue;
    int j = -1;
    for (int i = 0; i < g.n_res; ++i) if (g.t[i].model == m) { j = i; break; }
    if (j < 0 && g.n_res >= RMAX) continue;                // no slot for a cold model
    float wait = g.t_avail_ms;
    if (j < 0) wait = wait + mi[m].load_ms;                // cold start: weight load
    const int br0 = (int)(rq.L < (uint32_t)T.B ? rq.L : (uint32_t)T.B) - 1;
    const int br1 = (j >= 0 && g.t[j].q[1] > 0) ? g.t[j].beta[1] + 1 : 0;
    if (br1 >= T.B) continue;
    // Ecur: energy of the GPU as it is now, at F_curr, slot-order sum (R:s4)
    float Ecur = 0.0f;
    for (int i = 0; i < g.n_res; ++i) {
      TenantEval te = tenant_eval(T, g.t[i], g.f_cur, g.t[i].sigma, false);
      Ecur = (i == 0) ? te.e : (Ecur + te.e);
    }
    for (int sg = 0; sg < smf; ++sg) {
      int f_req = -1;
      for (int phi = 0; phi < T.F; ++phi) {
        bool ok_co = true; float A = 0.0f;
        for (int i = 0; i < g.n_res; ++i) {
          TenantEval te = tenant_eval(T, g.t[i], phi, g.t[i].sigma, i == j);
          ok_co = ok_co && te.ok;
          A = (i == 0) ? te.e : (A + te.e);
        }
        Slot s0 = slot_eval(T, m, 0, phi, sg, br0 < 0 ? 0 : br0, rq.L, wait, rq.slo_ttft_ms);
        Slot s1 = slot_eval(T, m, 1, phi, sg, br1, O, 0.0f, rq.slo_tbt_ms);
        if (!(ok_co && s0.ok && s1.ok)) continue;
        float dE = (A + (s0.e + s1.e)) - Ecur;
        if (!(dE < INF)) continue;                         // overflowed energy = infeasible (R:s23)
        if (dE == 0.0f) dE = 0.0f;                         // -0 -> +0
        if (f_req < 0) f_req = phi;
        uint32_t flat = (uint32_t)((k * T.S + sg) * T.F + phi);
        if (!have || dE < bestE) {                         // strict <: first (lowest flat) wins ties
          have = true; bestE = dE; bestFlat = flat;
          best.gpu = k; best.sigma = (int16_t)sg; best.phi = (int16_t)phi;
          best.beta = (int16_t)br1; best.f_req = (int16_t)f_req;
          best.energy_mj = dE; best.ttft_ms = wait + s0.t;
          best.tbt_ms = T.LAT(m, 1, phi, sg, br1); best.flat = flat;
        }
      }
    }
  }
  (void)bestFlat;
  out = best;
}

// ------------------------------------------------------------------------------------------
// fs_dispatch: the paper's own three-phase dispatcher (Fig. 6), one operating point
// per GPU: S_k = SM_free (all free share units), f_k = F_curr.
//   Phase 1: GPU k is feasible iff the request, starting at T_avail with SM_free SMs,
//     meets its deadlines at F_curr (plus memory / slot eligibility as in fs_place_batch).
//   Phase 2 (Eq. 2-3): E^k = Power x Latency of the request's own prefill + decode
//     work at (f_k, S_k); k* = argmin E^k.  Near-ties: among feasible GPUs with
//     E^k <= fl(1.02*E_min) take the most free memory, then the largest SM_free, then lowest k.
//   Phase 3: no feasible GPU -> walk the GPUs in ascending T_avail (ties: lowest k),
//     evaluate at F_max (last frequency level), take the first feasible one.  Still none ->
//     scale out: gpu = -1 and the energy-optimal feasible frequency of a fresh, empty GPU
//     (all S units, wait = load_ms), "minimizing energy usage without violating SLOs".
// Output: Placement with f_req reused as the phase that decided (1 = F_curr, 2 = F_max retry,
// 3 = scale-out, -1 = nothing feasible even on a fresh GPU); flat = (k*S+sigma)*F+phi.
struct OwnEval { bool ok; float e, ttft, tbt; };
OwnEval own_eval(const Tables& T, const Request& rq, uint32_t O, int phi, int sg, int br1, float wait) {
  const int m = rq.model;
  const int br0 = (int)(rq.L < (uint32_t)T.B ? rq.L : (uint32_t)T.B) - 1;
  Slot s0 = slot_eval(T, m, 0, phi, sg, br0 < 0 ? 0 : br0, rq.L, wait, rq.slo_ttft_ms);
  Slot s1 = slot_eval(T, m, 1, phi, sg, br1, O, 0.0f, rq.slo_tbt_ms);
  float e = s0.e + s1.e;
  return {s0.ok && s1.ok && e < INF, e, wait + s0.t, T.LAT(m, 1, phi, sg, br1)};
}

void dispatch_one(const Tables& T, const ModelInfo* mi, const GpuState* gs, int K,
                  const Request& rq, Placement& out) {
  const int m = rq.model;
  const uint32_t O = (21u * rq.o_pred + 19u) / 20u;
  const float mem = (float)(rq.L + O) * mi[m].kv_mb_per_token;
  Placement best{}; best.gpu = -1; best.sigma = best.phi = best.beta = best.f_req = -1;
  best.energy_mj = INF; best.ttft_ms = INF; best.tbt_ms = INF; best.flat = 0xFFFFFFFFu;
  struct Cand { bool elig; int smf, br1; float wait; };
  std::vector<Cand> cd(K);
  for (int k = 0; k < K; ++k) {                            // eligibility, as in fs_place_batch
    const GpuState& g = gs[k]; Cand c{false, 0, 0, 0.0f};
    if (g.n_res >= 1 && mem <= g.mem_free_mb) {
      c.smf = sm_free_of(g, T.S);
      int j = -1;
      for (int i = 0; i < g.n_res; ++i) if (g.t[i].model == m) { j = i; break; }
      c.wait = g.t_avail_ms;
      if (j < 0) c.wait = c.wait + mi[m].load_ms;
      c.br1 = (j >= 0 && g.t[j].q[1] > 0) ? g.t[j].beta[1] + 1 : 0;
      c.elig = c.smf >= 1 && (j >= 0 || g.n_res < RMAX) && c.br1 < T.B;
    }
    cd[k] = c;
  }
  auto fill = [&](int k, int phi, const OwnEval& ev, int phase) {
    best.gpu = k; best.sigma = (int16_t)(cd[k].smf - 1); best.phi = (int16_t)phi;
    best.beta = (int16_t)cd[k].br1; best.f_req = (int16_t)phase; best.energy_mj = ev.e;
    best.ttft_ms = ev.ttft; best.tbt_ms = ev.tbt;
    best.flat = (uint32_t)((k * T.S + cd[k].smf - 1) * T.F + phi);
  };
  // Phase 1 + 2 at F_curr
  float emin = INF;
  for (int k = 0; k < K; ++k) if (cd[k].elig) {
    OwnEval ev = own_eval(T, rq, O, gs[k].f_cur, cd[k].smf - 1, cd[k].br1, cd[k].wait);
    if (ev.ok && ev.e < emin) emin = ev.e;
  }
  if (emin < INF) {
    const float band = 1.02f * emin;
    int bk = -1;
    for (int k = 0; k < K; ++k) if (cd[k].elig) {
      OwnEval ev = own_eval(T, rq, O, gs[k].f_cur, cd[k].smf - 1, cd[k].br1, cd[k].wait);
      if (!(ev.ok && ev.e <= band)) continue;
      if (bk < 0 || gs[k].mem_free_mb > gs[bk].mem_free_mb ||
          (gs[k].mem_free_mb == gs[bk].mem_free_mb && cd[k].smf > cd[bk].smf)) {
        bk = k; fill(k, gs[k].f_cur, ev, 1);
      }
    }
    out = best; return;
  }
  // Phase 3: F_max retry in T_avail order
  {
    int bk = -1; OwnEval bev{};
    for (int k = 0; k < K; ++k) if (cd[k].elig) {
      OwnEval ev = own_eval(T, rq, O, T.F - 1, cd[k].smf - 1, cd[k].br1, cd[k].wait);
      if (ev.ok && (bk < 0 || gs[k].t_avail_ms < gs[bk].t_avail_ms)) { bk = k; bev = ev; }
    }
    if (bk >= 0) { fill(bk, T.F - 1, bev, 2); out = best; return; }
  }
  // scale-out: best frequency of a fresh GPU
  for (int phi = 0; phi < T.F; ++phi) {
    OwnEval ev = own_eval(T, rq, O, phi, T.S - 1, 0, mi[m].load_ms);
    if (ev.ok && ev.e < best.energy_mj) {
      best.sigma = (int16_t)(T.S - 1); best.phi = (int16_t)phi; best.beta = 0; best.f_req = 3;
      best.energy_mj = ev.e; best.ttft_ms = ev.ttft; best.tbt_ms = ev.tbt;
    }
  }
  out = best;
}

// The sequential commit pass between the requests of one batch (reading R:s34 of
// P:214-218): the requests are dispatched one after the other, in the caller's order, each against the
// state the previous ones left.  A request sent to GPU k (phase 1 or 2) starts at its wait time with ALL
// of SM_free_k units (Eq. 2: Latency(f_k, S_k, ...)) and holds them until it completes, so
//   T_avail_k  <- fl(ttft + t_dec),  t_dec = fl(ceil(O/(beta+1)) * LAT1)   the earliest time the next
//                                                                request can start there (SM_free as polled)
//   mem_free_k <- fl(mem_free_k - Req_mem)      the memory stays reserved until the next poll
//   F_curr_k   <- phi                           (phase 2 raised the clock to F_max; phase 1 leaves it)
// A scale-out decision (gpu = -1) changes no record: activating a GPU is the caller's action.
// The resident models of a GPU are those of the last poll (a second request of a model that was cold is
// charged load_ms again: never an under-estimate of a TTFT).
void dispatch_commit(const Tables& T, const ModelInfo* mi, GpuState* gs, int K, const Request* rq, int R,
                     Placement* out) {
  for (int r = 0; r < R; ++r) {
    dispatch_one(T, mi, gs, K, rq[r], out[r]);
    const Placement& p = out[r];
    if (p.gpu < 0) continue;
    const uint32_t O = (21u * rq[r].o_pred + 19u) / 20u;
    const float mem = (float)(rq[r].L + O) * mi[rq[r].model].kv_mb_per_token;
    float tdec = 0.0f;
    if (O > 0) {
      const uint32_t n = (uint32_t)p.beta + 1u;
      tdec = (float)((O + n - 1u) / n) * p.tbt_ms;          // tbt_ms = LAT1 at the chosen point
    }
    GpuState& g = gs[p.gpu];
    g.t_avail_ms = p.ttft_ms + tdec;
    g.mem_free_mb = g.mem_free_mb - mem;
    g.f_cur = p.phi;
  }
}

// ------------------------------------------------------------------------------------------
// Algorithm 1, Phase 1: per active LLM, from its average input / output length:
//   (SM_p, F_p), (SM_d, F_d) = the LUT configurations that minimise the prefill / decode energy
//   while meeting the TTFT / TBT SLO (ties: lowest phi, then lowest sigma); T_p, T_d, P_p, P_d there;
//   SM_l = (SM_p*T_p + SM_d*T_d) / (T_p + T_d)                                   (Eq. 8)
//   l.S  = ceil(SM_l) share units;  l.F = the frequency that minimises the LLM's total energy at
//   l.S units with both SLOs met (CalcFreq, Alg. 1 l.4; lowest phi on ties);
//   M_l  = Weights + N_conc * Size_KV,  N_conc = lambda * W (Little's law), W = T_p + T_d at
//   (l.S, l.F), Size_KV = (avg_in + avg_out) * kv_mb_per_token.
// One sequence per decode step (batch bucket 0), the prefill batch bucket as in fs_place_batch.
struct Llm { int32_t model; uint32_t avg_in, avg_out; float slo_ttft_ms, slo_tbt_ms, lambda_rps; uint32_t pad[2]; };
struct LlmProfile {
  int16_t sigma_p, phi_p, sigma_d, phi_d; float t_p_ms, t_d_ms, p_p_w, p_d_w;
  float sm_units; int16_t need_units, phi_l; float t_l_ms, e_l_mj, mem_mb; uint32_t pad;
};
static_assert(sizeof(Llm) == 32 && sizeof(LlmProfile) == 48, "layout");

void llm_profile_one(const Tables& T, const ModelInfo* mi, const Llm& l, LlmProfile& o) {
  const int m = l.model;
  const uint32_t L = l.avg_in, O = l.avg_out;
  const int br0 = (int)(L < (uint32_t)T.B ? L : (uint32_t)T.B) - 1;
  std::memset(&o, 0, sizeof(o));
  o.sigma_p = o.phi_p = o.sigma_d = o.phi_d = o.need_units = o.phi_l = -1;
  o.t_p_ms = o.t_d_ms = o.p_p_w = o.p_d_w = o.sm_units = o.t_l_ms = o.e_l_mj = o.mem_mb = INF;
  float bp = INF, bd = INF;
  for (int phi = 0; phi < T.F; ++phi)
    for (int sg = 0; sg < T.S; ++sg) {
      Slot p = slot_eval(T, m, 0, phi, sg, br0 < 0 ? 0 : br0, L, 0.0f, l.slo_ttft_ms);
      if (p.ok && p.e < bp) {
        bp = p.e; o.sigma_p = (int16_t)sg; o.phi_p = (int16_t)phi; o.t_p_ms = p.t;
        o.p_p_w = L ? T.POW(m, 0, phi, sg, br0) : 0.0f;
      }
      Slot d = slot_eval(T, m, 1, phi, sg, 0, O, 0.0f, l.slo_tbt_ms);
      if (d.ok && d.e < bd) {
        bd = d.e; o.sigma_d = (int16_t)sg; o.phi_d = (int16_t)phi; o.t_d_ms = d.t;
        o.p_d_w = O ? T.POW(m, 1, phi, sg, 0) : 0.0f;
      }
    }
  if (o.phi_p < 0 || o.phi_d < 0) return;                 // one phase cannot meet its SLO anywhere
  const float tsum = o.t_p_ms + o.t_d_ms;
  o.sm_units = tsum > 0.0f ? (((float)(o.sigma_p + 1) * o.t_p_ms + (float)(o.sigma_d + 1) * o.t_d_ms) / tsum) : 1.0f;
  int need = (int)std::ceil(o.sm_units);
  if (need < 1) need = 1;
  if (need > T.S) need = T.S;
  o.need_units = (int16_t)need;
  float be = INF;
  for (int phi = 0; phi < T.F; ++phi) {
    Slot p = slot_eval(T, m, 0, phi, need - 1, br0 < 0 ? 0 : br0, L, 0.0f, l.slo_ttft_ms);
    Slot d = slot_eval(T, m, 1, phi, need - 1, 0, O, 0.0f, l.slo_tbt_ms);
    const float e = p.e + d.e;
    if (p.ok && d.ok && e < be) { be = e; o.phi_l = (int16_t)phi; o.t_l_ms = p.t + d.t; o.e_l_mj = e; }
  }
  if (o.phi_l < 0) return;
  const float nconc = l.lambda_rps * (o.t_l_ms / 1000.0f);
  const float kvsize = (float)(L + O) * mi[m].kv_mb_per_token;
  o.mem_mb = mi[m].weights_mb + nconc * kvsize;
}

// Energy Waste Ratio (Eq. 5-7): F_g = highest preferred frequency among the LLMs on GPU g,
//   E_waste = sum t_l (F_g^3 - F_l^3),  E_optimal = sum t_l F_l^3,  EWR = E_waste / E_optimal.
// Plain left-to-right sums in binary64 over the LLMs in index order; gpu < 0 = not placed.
void ewr_all(int n, const int32_t* gpu_of, const float* f_mhz, const float* t_ms, int K, float* fg, double out[3]) {
  for (int g = 0; g < K; ++g) fg[g] = 0.0f;
  for (int l = 0; l < n; ++l) if (gpu_of[l] >= 0 && f_mhz[l] > fg[gpu_of[l]]) fg[gpu_of[l]] = f_mhz[l];
  double waste = 0.0, opt = 0.0;
  for (int l = 0; l < n; ++l) {
    if (gpu_of[l] < 0) continue;
    const double F = fg[gpu_of[l]], f = f_mhz[l], t = t_ms[l];
    waste += t * (F * F * F - f * f * f);
    opt += t * (f * f * f);
  }
  out[0] = waste; out[1] = opt; out[2] = opt > 0.0 ? waste / opt : 0.0;
}

// ------------------------------------------------------------------------------------------
// Algorithm 1, phases 2-3 (prose P:341-357): capacity planning by Best-Fit-Decreasing and the
// EWR-minimising placement loop.  Readings: BFD sorts by decreasing size (ties: lower
// index), puts an item into the open bin with the least remaining room that still fits (ties: lower
// bin), else opens a bin; an LLM that exceeds a whole GPU is left unplaced (gpu = -1).  Phase 3 walks the
// LLMs in ascending l.F (ties: lower index).  g.freq = highest l.F on g; the distance of an EMPTY GPU is
// +INF (it is the last resort, so that similar frequencies group on the same GPU); ties: lower GPU.
//   Target = closest GPU, Candidate = second closest.   Fits = SM units and memory both fit.
//   1. Fits(target, l): assign.                                   (direct placement)
//   2. else l_out = resident of target with the lowest l.F (ties: lower index); if Fits(cand, l_out) and
//      Fits(target - l_out, l) and E_swap < E_curr: move l_out to cand, assign l to target, where
//      E_curr = waste(target + l) + waste(cand), E_swap = waste(target - l_out + l) + waste(cand + l_out),
//      waste(R) = sum_{r in R} t_r (F_R^3 - F_r^3), F_R = max F_r, binary64, residents in the order they
//      joined, the hypothetical newcomer last.                    (EWR-driven swap, Alg. 1 l.16-21)
//   3. else if Fits(cand, l): assign to cand (l.23-24); else the closest other GPU that fits (fallback,
//      P:357); else activate a new GPU (l.26-27).
struct PlanLlm { int32_t need_units; float mem_mb, f_mhz, t_ms; };
static_assert(sizeof(PlanLlm) == 16, "layout");

int bfd_units(const PlanLlm* L, int n, int cap) {
  std::vector<int> order; for (int i = 0; i < n; ++i) if (L[i].need_units <= cap) order.push_back(i);
  for (size_t a = 1; a < order.size(); ++a) {              // insertion sort, decreasing, stable
    int x = order[a]; int b = (int)a - 1;
    while (b >= 0 && L[order[b]].need_units < L[x].need_units) { order[b + 1] = order[b]; --b; }
    order[b + 1] = x;
  }
  std::vector<int> rem;
  for (int i : order) {
    int best = -1;
    for (size_t g = 0; g < rem.size(); ++g)
      if (rem[g] >= L[i].need_units && (best < 0 || rem[g] < rem[best])) best = (int)g;
    if (best < 0) { rem.push_back(cap); best = (int)rem.size() - 1; }
    rem[best] -= L[i].need_units;
  }
  return (int)rem.size();
}
int bfd_mem(const PlanLlm* L, int n, float cap) {
  std::vector<int> order; for (int i = 0; i < n; ++i) if (L[i].mem_mb <= cap) order.push_back(i);
  for (size_t a = 1; a < order.size(); ++a) {
    int x = order[a]; int b = (int)a - 1;
    while (b >= 0 && L[order[b]].mem_mb < L[x].mem_mb) { order[b + 1] = order[b]; --b; }
    order[b + 1] = x;
  }
  std::vector<float> rem;
  for (int i : order) {
    int best = -1;
    for (size_t g = 0; g < rem.size(); ++g)
      if (rem[g] >= L[i].mem_mb && (best < 0 || rem[g] < rem[best])) best = (int)g;
    if (best < 0) { rem.push_back(cap); best = (int)rem.size() - 1; }
    rem[best] = rem[best] - L[i].mem_mb;
  }
  return (int)rem.size();
}

struct PlanGpu { int sm_left; float mem_left; std::vector<int> res; };
float plan_freq(const PlanLlm* L, const PlanGpu& g) {
  float f = 0.0f; for (int r : g.res) if (L[r].f_mhz > f) f = L[r].f_mhz; return f;
}
// waste of the residents of g without `skip` (-1: none) plus `extra` (-1: none), extra last
double plan_waste(const PlanLlm* L, const PlanGpu& g, int skip, int extra) {
  float F = 0.0f;
  for (int r : g.res) if (r != skip && L[r].f_mhz > F) F = L[r].f_mhz;
  if (extra >= 0 && L[extra].f_mhz > F) F = L[extra].f_mhz;
  const double F3 = (double)F * F * F;
  double w = 0.0;
  for (int r : g.res) if (r != skip) { const double f = L[r].f_mhz; w += (double)L[r].t_ms * (F3 - f * f * f); }
  if (extra >= 0) { const double f = L[extra].f_mhz; w += (double)L[extra].t_ms * (F3 - f * f * f); }
  return w;
}

void replace_plan(const PlanLlm* L, int n, int s_eff, float m_eff, int32_t* gpu_of, int32_t summary[4]) {
  const int n_sm = bfd_units(L, n, s_eff), n_mem = bfd_mem(L, n, m_eff);
  const int n_min = n_sm > n_mem ? n_sm : n_mem;
  std::vector<PlanGpu> G(n_min, PlanGpu{s_eff, m_eff, {}});
  std::vector<int> order(n);
  for (int i = 0; i < n; ++i) { order[i] = i; gpu_of[i] = -1; }
  for (int a = 1; a < n; ++a) {                             // ascending l.F, stable
    int x = order[a], b = a - 1;
    while (b >= 0 && L[order[b]].f_mhz > L[x].f_mhz) { order[b + 1] = order[b]; --b; }
    order[b + 1] = x;
  }
  auto fits = [&](const PlanGpu& g, int l, int freed_units, float freed_mem, bool freed) {
    const int sm = g.sm_left + freed_units;
    const float mem = freed ? (g.mem_left + freed_mem) : g.mem_left;
    return L[l].need_units <= sm && L[l].mem_mb <= mem;
  };
  auto put = [&](int g, int l) {
    G[g].sm_left -= L[l].need_units; G[g].mem_left = G[g].mem_left - L[l].mem_mb; G[g].res.push_back(l); gpu_of[l] = g;
  };
  for (int l : order) {
    if (L[l].need_units > s_eff || !(L[l].mem_mb <= m_eff)) continue;       // exceeds a whole GPU
    auto dist = [&](int g) { return G[g].res.empty() ? INF : std::fabs(plan_freq(L, G[g]) - L[l].f_mhz); };
    int tgt = -1, cand = -1;
    for (int g = 0; g < (int)G.size(); ++g) if (tgt < 0 || dist(g) < dist(tgt)) tgt = g;
    for (int g = 0; g < (int)G.size(); ++g) if (g != tgt && (cand < 0 || dist(g) < dist(cand))) cand = g;
    bool done = false;
    if (tgt >= 0 && fits(G[tgt], l, 0, 0.0f, false)) { put(tgt, l); done = true; }
    if (!done && tgt >= 0 && cand >= 0 && !G[tgt].res.empty()) {
      int lo = -1;
      for (int r : G[tgt].res) if (lo < 0 || L[r].f_mhz < L[lo].f_mhz || (L[r].f_mhz == L[lo].f_mhz && r < lo)) lo = r;
      const double e_curr = plan_waste(L, G[tgt], -1, l) + plan_waste(L, G[cand], -1, -1);
      const double e_swap = plan_waste(L, G[tgt], lo, l) + plan_waste(L, G[cand], -1, lo);
      if (fits(G[cand], lo, 0, 0.0f, false) && fits(G[tgt], l, L[lo].need_units, L[lo].mem_mb, true) && e_swap < e_curr) {
        PlanGpu& t = G[tgt];
        t.sm_left += L[lo].need_units; t.mem_left = t.mem_left + L[lo].mem_mb;
        for (size_t x = 0; x < t.res.size(); ++x) if (t.res[x] == lo) { t.res.erase(t.res.begin() + x); break; }
        put(cand, lo); put(tgt, l); done = true;
      }
    }
    if (!done && cand >= 0 && fits(G[cand], l, 0, 0.0f, false)) { put(cand, l); done = true; }
    if (!done) {
      int fb = -1;
      for (int g = 0; g < (int)G.size(); ++g)
        if (g != tgt && g != cand && fits(G[g], l, 0, 0.0f, false) && (fb < 0 || dist(g) < dist(fb))) fb = g;
      if (fb >= 0) { put(fb, l); done = true; }
    }
    if (!done) { G.push_back(PlanGpu{s_eff, m_eff, {}}); put((int)G.size() - 1, l); }
  }
  summary[0] = n_sm; summary[1] = n_mem; summary[2] = n_min; summary[3] = (int)G.size();
}

// ------------------------------------------------------------------------------------------
// Appendix E: transmission plan and selective request migration.
//   e_uv = Bytes(u -> v) / BW(u, v); minimum-cost assignment of sources to destinations by the
//   Kuhn-Munkres algorithm.  Costs are taken in whole microseconds, c_uv = rint(fl(fl(bytes_u / bw_uv) * 1000))
//   with bytes in MB and bw in MB/ms (reading s33), so the optimum is an exact integer.
//   Shortest-augmenting-path form with row / column potentials; ties: lowest column.
void assign_min_cost(int n, const float* bytes_mb, const float* bw, int32_t* dst_of, int64_t* total_us) {
  const int64_t BIG = (int64_t)1 << 60;
  auto cost = [&](int u, int v) { return (int64_t)std::llrint((bytes_mb[u] / bw[(size_t)u * n + v]) * 1000.0f); };
  std::vector<int64_t> pu(n + 1, 0), pv(n + 1, 0), minv(n + 1);
  std::vector<int> p(n + 1, 0), way(n + 1, 0);               // p[j] = row matched to column j (1-based, 0 = none)
  for (int i = 1; i <= n; ++i) {
    p[0] = i; int j0 = 0;
    std::vector<char> used(n + 1, 0);
    for (int j = 0; j <= n; ++j) minv[j] = BIG;
    do {
      used[j0] = 1;
      const int i0 = p[j0]; int64_t delta = BIG; int j1 = 0;
      for (int j = 1; j <= n; ++j) if (!used[j]) {
        const int64_t cur = cost(i0 - 1, j - 1) - pu[i0] - pv[j];
        if (cur < minv[j]) { minv[j] = cur; way[j] = j0; }
        if (minv[j] < delta) { delta = minv[j]; j1 = j; }
      }
      for (int j = 0; j <= n; ++j) {
        if (used[j]) { pu[p[j]] += delta; pv[j] -= delta; } else minv[j] -= delta;
      }
      j0 = j1;
    } while (p[j0] != 0);
    do { const int j1 = way[j0]; p[j0] = p[j1]; j0 = j1; } while (j0);
  }
  int64_t tot = 0;
  for (int j = 1; j <= n; ++j) { dst_of[p[j] - 1] = j - 1; }
  for (int u = 0; u < n; ++u) tot += cost(u, dst_of[u]);
  *total_us = tot;
}

// Per in-flight request: KV is transferred iff that is faster than recomputing it on the
// destination; the request migrates iff its remaining computation on the source exceeds the migration
// time; otherwise it finishes in place.  out: bit 0 = migrate, bit 1 = transfer KV (else tokens only).
struct MigReq { float remaining_ms, tokens_mb, kv_mb, bw_mb_per_ms, recompute_ms; uint32_t pad[3]; };
static_assert(sizeof(MigReq) == 32, "layout");
void migration_select(int r, const MigReq* q, uint8_t* out, float* mig_ms) {
  for (int i = 0; i < r; ++i) {
    const float kv_tx = q[i].kv_mb / q[i].bw_mb_per_ms;
    const bool kv = kv_tx < q[i].recompute_ms;
    const float t = (q[i].tokens_mb / q[i].bw_mb_per_ms) + (kv ? kv_tx : q[i].recompute_ms);
    mig_ms[i] = t;
    out[i] = (uint8_t)((q[i].remaining_ms > t ? 1 : 0) | (kv ? 2 : 0));
  }
}

// ------------------------------------------------------------------------------------------
// fs_local_config: frequency sweep with per-task SM allocation (Fig. 8 step 3,
// P:206-210); batching P:248; objective R:s8; split domain R:s9; one beta per slot R:s10.
// Hierarchical definition: best beta per slot, then tenant sums, then the argmin.
struct SlotBest { float g; int beta; float e; float pw; };

SlotBest slot_search(const Tables& T, const Tenant& t, int p, int phi, int sigma, bool obj_power) {
  if (t.q[p] == 0) return {0.0f, 0, 0.0f, 0.0f};
  SlotBest b{INF, 0, 0.0f, 0.0f};
  int nb = (int)(t.q[p] < (uint32_t)T.B ? t.q[p] : (uint32_t)T.B);
  for (int beta = 0; beta < nb; ++beta) {
    Slot s = slot_eval(T, t.model, p, phi, sigma, beta, t.q[p], 0.0f, t.slo_ms[p]);
    if (!s.ok) continue;
    float pw = T.POW(t.model, p, phi, sigma, beta);
    float cost = obj_power ? pw : s.e;
    if (cost < b.g) { b.g = cost; b.beta = beta; b.e = s.e; b.pw = pw; }
  }
  return b;
}

uint64_t binom(int n, int k) {
  if (k < 0 || k > n) return 0;
  uint64_t r = 1;
  for (int i = 1; i <= k; ++i) r = r * (uint64_t)(n - k + i) / (uint64_t)i;
  return r;
}

void local_one(const Tables& T, const GpuState& g, uint32_t flags, LocalCfg& out) {
  const bool obj_power = flags & 1u, minsm = flags & 2u;
  std::memset(&out, 0, sizeof(out));
  out.phi = -1; out.f_req = -1; out.flat = 0xFFFFFFFFu;
  const int n = g.n_res;
  if (n < 1) { out.cost = 0.0f; return; }
  out.cost = INF; out.energy_mj = INF; out.power_w = INF;
  if (n > T.S) return;
  const int F = T.F, S = T.S;
  // G_i[phi][sigma] and the slot minima behind it
  std::vector<SlotBest> sb((size_t)n * 2 * F * S);
  std::vector<float> G((size_t)n * F * S);
  auto SB = [&](int i, int p, int phi, int sg) -> SlotBest& { return sb[(((size_t)i * 2 + p) * F + phi) * S + sg]; };
  auto GG = [&](int i, int phi, int sg) -> float& { return G[((size_t)i * F + phi) * S + sg]; };
  for (int i = 0; i < n; ++i)
    for (int phi = 0; phi < F; ++phi)
      for (int sg = 0; sg < S; ++sg) {
        SB(i, 0, phi, sg) = slot_search(T, g.t[i], 0, phi, sg, obj_power);
        SB(i, 1, phi, sg) = slot_search(T, g.t[i], 1, phi, sg, obj_power);
        GG(i, phi, sg) = SB(i, 0, phi, sg).g + SB(i, 1, phi, sg).g;
      }
  bool have = false; float bestC = INF; int bphi = -1; int bsig[RMAX] = {0, 0, 0, 0}; uint32_t bflat = 0;
  int f_req = -1;
  if (minsm) {
    // the paper's rule: per frequency, each task's minimum SM meeting its deadline; sum <= budget
    for (int phi = 0; phi < F; ++phi) {
      int sig[RMAX]; bool all = true; int tot = 0;
      for (int i = 0; i < n && all; ++i) {
        sig[i] = -1;
        for (int sg = 0; sg < S; ++sg) if (GG(i, phi, sg) < INF) { sig[i] = sg; break; }
        if (sig[i] < 0) all = false; else tot += sig[i] + 1;
      }
      if (!all || tot > S) continue;                      // "<= budget": Fig. 8 accepts 100 % (R:s7)
      float C = 0.0f;
      for (int i = 0; i < n; ++i) C = (i == 0) ? GG(i, phi, sig[i]) : (C + GG(i, phi, sig[i]));
      if (!(C < INF)) continue;
      if (f_req < 0) f_req = phi;
      if (!have || C < bestC) { have = true; bestC = C; bphi = phi; bflat = (uint32_t)phi; for (int i = 0; i < n; ++i) bsig[i] = sig[i]; }
    }
  } else {
    const uint64_t NS = binom(S - 1, n - 1);
    for (int phi = 0; phi < F; ++phi) {
      // all compositions of S into n positive parts, lexicographic with sigma_0 most significant
      int sig[RMAX] = {0, 0, 0, 0};
      uint64_t rank = 0;
      // plain nested loops over (sigma_0..sigma_3), keeping the tuples that sum to S (n <= 4)
      for (int s0 = 0; s0 < S; ++s0) {
        if (n == 1) { if (s0 + 1 != S) continue; }
        for (int s1 = 0; s1 < (n >= 2 ? S : 1); ++s1) {
          if (n == 2) { if (s0 + 1 + s1 + 1 != S) continue; }
          for (int s2 = 0; s2 < (n >= 3 ? S : 1); ++s2) {
            if (n == 3) { if (s0 + s1 + s2 + 3 != S) continue; }
            for (int s3 = 0; s3 < (n >= 4 ? S : 1); ++s3) {
              if (n == 4) { if (s0 + s1 + s2 + s3 + 4 != S) continue; }
              sig[0] = s0; sig[1] = s1; sig[2] = s2; sig[3] = s3;
              float C = 0.0f;
              for (int i = 0; i < n; ++i) C = (i == 0) ? GG(i, phi, sig[i]) : (C + GG(i, phi, sig[i]));
              uint64_t this_rank = rank++;
              if (!(C < INF)) continue;
              if (f_req < 0) f_req = phi;
              if (!have || C < bestC) {
                have = true; bestC = C; bphi = phi; bflat = (uint32_t)((uint64_t)phi * NS + this_rank);
                for (int i = 0; i < n; ++i) bsig[i] = sig[i];
              }
            }
          }
        }
      }
    }
  }
  if (!have) return;
  out.phi = (int16_t)bphi; out.f_req = (int16_t)f_req; out.cost = bestC; out.flat = bflat;
  float E = 0.0f, PW = 0.0f;
  for (int i = 0; i < n; ++i) {
    const SlotBest& a = SB(i, 0, bphi, bsig[i]); const SlotBest& b = SB(i, 1, bphi, bsig[i]);
    out.sigma[i] = (uint8_t)bsig[i]; out.beta[i][0] = (uint8_t)a.beta; out.beta[i][1] = (uint8_t)b.beta;
    float ei = a.e + b.e, pi = a.pw + b.pw;
    E = (i == 0) ? ei : (E + ei); PW = (i == 0) ? pi : (PW + pi);
  }
  out.energy_mj = E; out.power_w = PW;
}

// ------------------------------------------------------------------------------------------
// fs_consolidate: drain-one-source scoring over all GPU pairs (R:s17).  Per-tenant minimum
// feasible share per frequency (P:252 rule (1)), 5 % margin on SMs and memory,
// idle power vs migration energy.
struct GpuAgg { std::vector<int> need; std::vector<float> E; float mem; float Cstar; int n; };

void consolidate_all(const Tables& T, const ModelInfo* mi, const GpuState* gs, int K,
                     float p_idle_w, float horizon_ms, float mem_cap_mb, int delta_pct,
                     ConsolOut* out, int nthreads) {
  const int F = T.F, S = T.S;
  const int NEED_INF = 1 << 20;
  const int S_eff = (S * (100 - delta_pct)) / 100;
  const float M_eff = (mem_cap_mb * (float)(100 - delta_pct)) / 100.0f;
  std::vector<GpuAgg> agg(K);
  for (int g = 0; g < K; ++g) {
    GpuAgg& a = agg[g]; a.n = gs[g].n_res; a.need.assign(F, NEED_INF); a.E.assign(F, INF); a.mem = 0.0f; a.Cstar = INF;
    if (a.n < 1) continue;
    for (int i = 0; i < a.n; ++i) a.mem = (i == 0) ? gs[g].t[i].mem_used_mb : (a.mem + gs[g].t[i].mem_used_mb);
    for (int phi = 0; phi < F; ++phi) {
      int need = 0; float E = 0.0f; bool all = true;
      for (int i = 0; i < a.n && all; ++i) {
        int smin = -1; float ei = INF;
        for (int sg = 0; sg < S; ++sg) {
          TenantEval te = tenant_eval(T, gs[g].t[i], phi, sg, false);
          if (te.ok) { smin = sg; ei = te.e; break; }
        }
        if (smin < 0) { all = false; break; }
        need += smin + 1; E = (i == 0) ? ei : (E + ei);
      }
      if (all) { a.need[phi] = need; a.E[phi] = E; }
      if (all && need <= S_eff && E < a.Cstar) a.Cstar = E;   // lowest phi on ties
    }
  }
  auto work = [&](int a0, int a1) {
    for (int a = a0; a < a1; ++a) {
      ConsolOut o; o.dst = -1; o.phi = -1; o.score_mj = INF; o.saving_mj = -INF;
      const GpuAgg& A = agg[a];
      if (A.n >= 1) {
        bool have = false;
        for (int b = 0; b < K; ++b) {
          const GpuAgg& Bg = agg[b];
          if (b == a || Bg.n < 1) continue;
          if (A.n + Bg.n > RMAX) continue;
          if (!((A.mem + Bg.mem) <= M_eff)) continue;
          if (!(Bg.Cstar < INF)) continue;
          float Cab = INF; int phis = -1;
          for (int phi = 0; phi < F; ++phi) {
            if (A.need[phi] + Bg.need[phi] > S_eff) continue;
            float e = Bg.E[phi] + A.E[phi];
            if (e < Cab) { Cab = e; phis = phi; }
          }
          if (phis < 0) continue;
          float score = Cab - Bg.Cstar;
          if (!have || score < o.score_mj) { have = true; o.dst = b; o.phi = phis; o.score_mj = score; }
        }
        if (have) {
          float mig = 0.0f;
          for (int i = 0; i < A.n; ++i) mig = (i == 0) ? mi[gs[a].t[i].model].mig_mj : (mig + mi[gs[a].t[i].model].mig_mj);
          o.saving_mj = ((p_idle_w * horizon_ms) + A.Cstar) - (o.score_mj + mig);
        }
      }
      out[a] = o;
    }
  };
  if (nthreads <= 1) { work(0, K); return; }
  std::vector<std::thread> th;
  for (int t = 0; t < nthreads; ++t) th.emplace_back(work, (int)((int64_t)K * t / nthreads), (int)((int64_t)K * (t + 1) / nthreads));
  for (auto& x : th) x.join();
}

template <class Fn> void par_for(int n, int nthreads, Fn fn) {
  if (nthreads <= 1) { for (int i = 0; i < n; ++i) fn(i); return; }
  std::vector<std::thread> th;
  for (int t = 0; t < nthreads; ++t)
    th.emplace_back([=]() { for (int i = t; i < n; i += nthreads) fn(i); });
  for (auto& x : th) x.join();
}

// ---- local scheduler steps 1-2: unified priority score and priority-based task batching ------
// Score_task = Latency(task) / (Slack_task - beta*Age_task), beta = 0 for decode, 1 for prefill
// (Eq. 4); Latency(task) = the LUT entry of the scheduling unit at the GPU's current
// frequency.  A task whose effective slack is used up (<= 0) is the most urgent: score +INF
// (reading s26).  Batching (Fig. 8 steps 1-2): walk the tasks in descending score
// (ties: lowest task index), admit a task iff its memory and SM share still fit, otherwise
// bypass it and go on.  Budgets: all S share units, the GPU's free memory.
struct Task { int16_t model; uint8_t phase, sigma, beta, p0[3]; float slack_ms, age_ms, mem_mb; uint32_t tag; };
struct TaskOut { float score, latency_ms; int32_t rank, admitted; };
static_assert(sizeof(Task) == 24 && sizeof(TaskOut) == 16, "layout");

void batch_one(const Tables& T, const GpuState& g, const Task* tk, int n, TaskOut* out) {
  std::vector<int> order(n);
  for (int i = 0; i < n; ++i) {
    const Task& t = tk[i];
    float lat = T.LAT(t.model, t.phase, g.f_cur, t.sigma, t.beta);
    float denom = (t.phase == 0) ? (t.slack_ms - t.age_ms) : t.slack_ms;
    out[i].latency_ms = lat;
    out[i].score = (denom > 0.0f) ? (lat / denom) : INF;
    order[i] = i;
  }
  // insertion sort: descending score, stable (lowest index first among equals)
  for (int a = 1; a < n; ++a) {
    int x = order[a], b = a - 1;
    while (b >= 0 && out[order[b]].score < out[x].score) { order[b + 1] = order[b]; --b; }
    order[b + 1] = x;
  }
  int sm_left = T.S; float mem_left = g.mem_free_mb;
  for (int pos = 0; pos < n; ++pos) {
    const int i = order[pos]; const Task& t = tk[i];
    out[i].rank = pos;
    const int need = (int)t.sigma + 1;
    if (need <= sm_left && t.mem_mb <= mem_left) {
      out[i].admitted = 1; sm_left -= need; mem_left = mem_left - t.mem_mb;
    } else out[i].admitted = 0;
  }
}

}  // namespace

extern "C" {

int fo_place_batch(int M, int F, int S, int B, const float* lat, const float* pow,
                   const void* models, int K, const void* states, int R, const void* reqs,
                   void* out, int nthreads) {
  Tables T{M, F, S, B, lat, pow};
  const ModelInfo* mi = (const ModelInfo*)models; const GpuState* gs = (const GpuState*)states;
  const Request* rq = (const Request*)reqs; Placement* o = (Placement*)out;
  par_for(R, nthreads, [&](int r) { place_one(T, mi, gs, K, rq[r], o[r]); });
  return 0;
}

int fo_dispatch(int M, int F, int S, int B, const float* lat, const float* pow,
                const void* models, int K, const void* states, int R, const void* reqs,
                void* out, int nthreads) {
  Tables T{M, F, S, B, lat, pow};
  const ModelInfo* mi = (const ModelInfo*)models; const GpuState* gs = (const GpuState*)states;
  const Request* rq = (const Request*)reqs; Placement* o = (Placement*)out;
  par_for(R, nthreads, [&](int r) { dispatch_one(T, mi, gs, K, rq[r], o[r]); });
  return 0;
}

// states is updated in place (the records after the last commit)
int fo_dispatch_commit(int M, int F, int S, int B, const float* lat, const float* pow,
                       const void* models, int K, void* states, int R, const void* reqs, void* out) {
  Tables T{M, F, S, B, lat, pow};
  dispatch_commit(T, (const ModelInfo*)models, (GpuState*)states, K, (const Request*)reqs, R, (Placement*)out);
  return 0;
}

int fo_llm_profile(int M, int F, int S, int B, const float* lat, const float* pow, const void* models,
                   int n, const void* llms, void* out, int nthreads) {
  Tables T{M, F, S, B, lat, pow};
  const ModelInfo* mi = (const ModelInfo*)models; const Llm* ll = (const Llm*)llms; LlmProfile* o = (LlmProfile*)out;
  par_for(n, nthreads, [&](int i) { llm_profile_one(T, mi, ll[i], o[i]); });
  return 0;
}

int fo_ewr(int n, const int32_t* gpu_of, const float* f_mhz, const float* t_ms, int K, float* fg, double* out3) {
  ewr_all(n, gpu_of, f_mhz, t_ms, K, fg, out3);
  return 0;
}

int fo_replace_plan(int n, const void* llms, int s_eff, float m_eff, int32_t* gpu_of, int32_t* summary4) {
  replace_plan((const PlanLlm*)llms, n, s_eff, m_eff, gpu_of, summary4);
  return 0;
}

int fo_assign(int n, const float* bytes_mb, const float* bw, int32_t* dst_of, int64_t* total_us) {
  assign_min_cost(n, bytes_mb, bw, dst_of, total_us);
  return 0;
}
int fo_migration_select(int r, const void* reqs, uint8_t* out, float* mig_ms) {
  migration_select(r, (const MigReq*)reqs, out, mig_ms);
  return 0;
}

int fo_local_config(int M, int F, int S, int B, const float* lat, const float* pow,
                    const void* states, int n, const int32_t* gpu_ids, uint32_t flags, void* out,
                    int nthreads) {
  Tables T{M, F, S, B, lat, pow};
  const GpuState* gs = (const GpuState*)states; LocalCfg* o = (LocalCfg*)out;
  par_for(n, nthreads, [&](int i) { local_one(T, gs[gpu_ids ? gpu_ids[i] : i], flags, o[i]); });
  return 0;
}

int fo_consolidate(int M, int F, int S, int B, const float* lat, const float* pow,
                   const void* models, int K, const void* states, float p_idle_w,
                   float horizon_ms, float mem_cap_mb, int delta_pct, void* out, int nthreads) {
  Tables T{M, F, S, B, lat, pow};
  consolidate_all(T, (const ModelInfo*)models, (const GpuState*)states, K, p_idle_w, horizon_ms,
                  mem_cap_mb, delta_pct, (ConsolOut*)out, nthreads);
  return 0;
}

// Exposed for the pins: the slot rule and the per-GPU co-resident summary (segmented max).
int fo_slot(int M, int F, int S, int B, const float* lat, const float* pow, int m, int p, int phi,
            int sigma, int beta, uint32_t q, float wait, float slo, float* t, float* e) {
  Tables T{M, F, S, B, lat, pow};
  Slot s = slot_eval(T, m, p, phi, sigma, beta, q, wait, slo);
  *t = s.t; *e = s.e; return s.ok ? 1 : 0;
}

// Lowest frequency index at which every co-resident of GPU g is feasible (-1 if none):
// the "device-wide operating point" lower bound, max over co-residents of each one's lowest
// feasible frequency when feasibility is monotone (R:s3).
int fo_gpu_freq_floor(int M, int F, int S, int B, const float* lat, const float* pow,
                      const void* state) {
  Tables T{M, F, S, B, lat, pow};
  const GpuState& g = *(const GpuState*)state;
  for (int phi = 0; phi < F; ++phi) {
    bool ok = true;
    for (int i = 0; i < g.n_res; ++i) ok = ok && tenant_eval(T, g.t[i], phi, g.t[i].sigma, false).ok;
    if (ok) return phi;
  }
  return -1;
}

// Per-tenant lowest feasible frequency (for the "max over co-residents" pin).
int fo_tenant_fmin(int M, int F, int S, int B, const float* lat, const float* pow,
                   const void* state, int i) {
  Tables T{M, F, S, B, lat, pow};
  const GpuState& g = *(const GpuState*)state;
  for (int phi = 0; phi < F; ++phi)
    if (tenant_eval(T, g.t[i], phi, g.t[i].sigma, false).ok) return phi;
  return -1;
}

// Steps 1-2 of the local scheduler for n GPUs; tasks of GPU i are tasks[off[i] .. off[i+1]).
int fo_batch_tasks(int M, int F, int S, int B, const float* lat, const float* pow,
                   const void* states, int n, const int32_t* gpu_ids, const int32_t* off,
                   const void* tasks, void* out, int nthreads) {
  Tables T{M, F, S, B, lat, pow};
  const GpuState* gs = (const GpuState*)states; const Task* tk = (const Task*)tasks; TaskOut* o = (TaskOut*)out;
  par_for(n, nthreads, [&](int i) {
    batch_one(T, gs[gpu_ids ? gpu_ids[i] : i], tk + off[i], off[i + 1] - off[i], o + off[i]);
  });
  return 0;
}

}  // extern "C"
