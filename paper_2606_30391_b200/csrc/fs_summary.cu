// fs_summary.cu — per-GPU co-resident summary, run by fs_set_gpu_state.
//
// For every GPU k and every frequency phi it evaluates each co-resident ("tenant") with the
// shared slot rule and reduces over the tenants of the GPU (the segment):
//   ok_co[k][v][phi] = AND_i ok_i(phi; bump = (i == v-1))      -> f_floor = lowest phi with ok
//   A[k][v][phi]     = ((e_0 + e_1) + ...) in slot order        (INF where !ok_co)
// for the variants v = 0 ("as is") and v = 1+j ("one more sequence joins tenant j's decode
// batch").  The shared frequency forces one operating point per device:
// f_floor is the max over co-residents of each one's lowest feasible frequency when feasibility
// is monotone, and is evaluated pointwise so it needs no monotonicity (R:s3).
// Also Ecur[k] (energy now, at F_curr), free SMs, and the decode bucket a joining request sees.
#include "fs_kernels.h"

namespace {

__device__ __forceinline__ bool state_valid(const fs_gpu_state& g, const FsDimsDev& d) {
  if (g.n_res < 0 || g.n_res > FS_RMAX) return false;
  if (g.n_res == 0) return true;
  if (g.f_cur < 0 || g.f_cur >= d.F) return false;
  int used = 0;
  for (int i = 0; i < g.n_res; ++i) {
    const fs_tenant& t = g.t[i];
    if (t.model < 0 || t.model >= d.M || t.sigma >= d.S || t.beta[0] >= d.B || t.beta[1] >= d.B ||
        t.q[0] >= (1u << 24) || t.q[1] >= (1u << 24))
      return false;
    used += t.sigma + 1;
  }
  return used <= d.S;
}

// the scan-order key of a compact record (see "scan order of the dense placement kernel" below)
__device__ __forceinline__ bool cold_capable(const FsGpuRec& r) {
  const int n = r.meta & 0xFF, smf = (r.meta >> 8) & 0xFF;
  return n >= 1 && n < FS_RMAX && smf >= 1 && r.a_min < FS_INF;
}
__device__ __forceinline__ float order_key(const FsGpuRec& r) {
  float d = cold_capable(r) ? __fsub_rn(r.a_min, r.e_cur) : FS_INF;
  return d == d ? d : FS_INF;
}
// one warp per GPU, lanes over phi
__global__ void __launch_bounds__(128) summary_kernel(FsView v, FsGpuInfo* __restrict__ ginfo,
                                                     float* __restrict__ gA,
                                                     FsGpuRec* __restrict__ grec,
                                                     float* __restrict__ gA0, float* __restrict__ okey) {
  const int lane = threadIdx.x & 31;
  const int k = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (k >= v.Kpad) return;
  const FsDimsDev d = v.d;
  if (k >= v.K) {            // padding rows of the staged arrays: never a candidate
    for (int phi = lane; phi < v.FT; phi += 32) gA0[(size_t)k * v.FT + phi] = FS_INF;
    if (lane == 0) {
      FsGpuRec r; r.t_avail_ms = r.mem_free_mb = r.e_cur = 0.f; r.meta = 0;
      for (int i = 0; i < FS_RMAX; ++i) r.model[i] = -1;
      r.a_min = FS_INF; r.k = 0;
      grec[k] = r; okey[k] = FS_INF;
    }
    return;
  }
  const fs_gpu_state g = v.states[k];
  const bool valid = state_valid(g, d);
  const int n = valid ? g.n_res : 0;
  float* A = gA + (size_t)k * FS_NVAR * d.F;
  int f_floor = -1; float a_min = FS_INF, ecur = 0.0f;
  // per tenant, independent of phi: plane offsets and rounds of the prefill slot, the decode slot as it is
  // and the decode slot with one more sequence (the integer divisions are done once, not per frequency)
  size_t o0[FS_RMAX], o1[FS_RMAX], o1b[FS_RMAX]; float r0[FS_RMAX], r1[FS_RMAX], r1b[FS_RMAX];
  bool has0[FS_RMAX], has1[FS_RMAX], bump_ok[FS_RMAX];
#pragma unroll
  for (int i = 0; i < FS_RMAX; ++i) {
    o0[i] = o1[i] = o1b[i] = 0; r0[i] = r1[i] = r1b[i] = 0.f; has0[i] = has1[i] = false; bump_ok[i] = true;
    if (i < n) {
      const fs_tenant& t = g.t[i];
      const int b1 = t.beta[1], b1b = b1 + (t.q[1] > 0 ? 1 : 0);
      has0[i] = t.q[0] > 0; has1[i] = t.q[1] > 0; bump_ok[i] = b1b < d.B;
      o0[i] = fs_plane(d, t.model, 0, t.beta[0]) + (size_t)t.sigma * d.F;
      o1[i] = fs_plane(d, t.model, 1, b1) + (size_t)t.sigma * d.F;
      o1b[i] = fs_plane(d, t.model, 1, min(b1b, d.B - 1)) + (size_t)t.sigma * d.F;
      r0[i] = __uint2float_rn(fs_ceil_div(t.q[0], t.beta[0] + 1u));
      r1[i] = __uint2float_rn(fs_ceil_div(t.q[1], b1 + 1u));
      r1b[i] = __uint2float_rn(fs_ceil_div(t.q[1], (uint32_t)min(b1b, d.B - 1) + 1u));
    }
  }
  for (int base = 0; base < d.F; base += 32) {
    const int phi = base + lane, pc = min(phi, d.F - 1);
    // every table entry of this frequency first (up to 24 independent loads in flight: the tables are
    // cold in L2 at this point of a step, and one miss after the other is what this kernel would wait for)
    float l0[FS_RMAX], p0[FS_RMAX], l1[FS_RMAX], p1[FS_RMAX], l1b[FS_RMAX], p1b[FS_RMAX];
#pragma unroll
    for (int i = 0; i < FS_RMAX; ++i) {
      l0[i] = p0[i] = l1[i] = p1[i] = l1b[i] = p1b[i] = 1.0f;
      if (i < n) {
        const float2 a = v.lpT[o0[i] + pc], b = v.lpT[o1[i] + pc], c = v.lpT[o1b[i] + pc];
        l0[i] = a.x; p0[i] = a.y; l1[i] = b.x; p1[i] = b.y; l1b[i] = c.x; p1b[i] = c.y;
      }
    }
    float e_plain[FS_RMAX], e_bump[FS_RMAX]; bool ok_plain[FS_RMAX], ok_bump[FS_RMAX];
    float esum = 0.0f;                                   // slot-order energy sum as it is (Ecur at F_curr)
#pragma unroll
    for (int i = 0; i < FS_RMAX; ++i) {
      e_plain[i] = e_bump[i] = 0.0f; ok_plain[i] = ok_bump[i] = true;
      if (i < n) {
        const fs_tenant& t = g.t[i];
        bool ok = true; float e0 = 0.0f, e1 = 0.0f, e1b = 0.0f; bool okb = true;
        if (has0[i]) { const FsSlot sl = fs_slot_f(0, l0[i], p0[i], r0[i], 0.0f, t.slo_ms[0]); ok = sl.ok; e0 = sl.e; }
        okb = ok;
        if (has1[i]) {
          const FsSlot sl = fs_slot_f(1, l1[i], p1[i], r1[i], 0.0f, t.slo_ms[1]); ok = ok && sl.ok; e1 = sl.e;
          const FsSlot sb = fs_slot_f(1, l1b[i], p1b[i], r1b[i], 0.0f, t.slo_ms[1]); okb = okb && sb.ok; e1b = sb.e;
        }
        e_plain[i] = __fadd_rn(e0, e1); ok_plain[i] = ok;
        if (has1[i]) { e_bump[i] = bump_ok[i] ? __fadd_rn(e0, e1b) : FS_INF; ok_bump[i] = bump_ok[i] && okb; }
        else { e_bump[i] = e_plain[i]; ok_bump[i] = ok; }
        esum = (i == 0) ? e_plain[i] : __fadd_rn(esum, e_plain[i]);
      }
    }
    if (n >= 1 && base == (g.f_cur & ~31)) ecur = __shfl_sync(0xffffffffu, esum, g.f_cur & 31);
    bool ok0 = false;
    if (phi < d.F) {
#pragma unroll
      for (int var = 0; var < FS_NVAR; ++var) {
        float acc = FS_INF; bool ok = (n >= 1) && (var <= n);
        if (ok) {
#pragma unroll
          for (int i = 0; i < FS_RMAX; ++i) {
            if (i < n) {
              const bool bump = (i == var - 1);
              const float e = bump ? e_bump[i] : e_plain[i];
              ok = ok && (bump ? ok_bump[i] : ok_plain[i]);
              acc = (i == 0) ? e : __fadd_rn(acc, e);   // slot-order sum
            }
          }
        }
        A[var * d.F + phi] = ok ? acc : FS_INF;
        if (var == 0) { ok0 = ok; gA0[(size_t)k * v.FT + phi] = ok ? acc : FS_INF; if (ok) a_min = fminf(a_min, acc); }
      }
    } else if (phi < v.FT) gA0[(size_t)k * v.FT + phi] = FS_INF;
    const unsigned m = __ballot_sync(0xffffffffu, ok0);
    if (f_floor < 0 && m) f_floor = base + __ffs(m) - 1;
  }
  for (int phi = (d.F + 31) / 32 * 32 + lane; phi < v.FT; phi += 32) gA0[(size_t)k * v.FT + phi] = FS_INF;   // stride padding
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a_min = fminf(a_min, __shfl_xor_sync(0xffffffffu, a_min, o));
  if (lane == 0) {
    FsGpuInfo gi;
    gi.t_avail_ms = g.t_avail_ms; gi.mem_free_mb = g.mem_free_mb;
    gi.n_res = n; gi.f_floor = f_floor; gi.f_cur = n ? g.f_cur : 0; gi._pad = 0;
    int used = 0;
    for (int i = 0; i < FS_RMAX; ++i) {
      if (i < n) {
        const fs_tenant& t = g.t[i];
        used += t.sigma + 1;
        gi.model[i] = t.model;
        const int b = (t.q[1] > 0) ? t.beta[1] + 1 : 0;
        gi.br1[i] = (int16_t)(b >= d.B ? -1 : b);
      } else { gi.model[i] = -1; gi.br1[i] = -1; }
    }
    gi.e_cur = ecur; gi.sm_free = n ? d.S - used : 0;
    ginfo[k] = gi;
    FsGpuRec r; r.t_avail_ms = gi.t_avail_ms; r.mem_free_mb = gi.mem_free_mb; r.e_cur = ecur;
    r.meta = (uint32_t)n | ((uint32_t)gi.sm_free << 8) | ((uint32_t)gi.f_cur << 16);
    for (int i = 0; i < FS_RMAX; ++i) r.model[i] = gi.model[i];
    r.a_min = a_min; r.k = (uint32_t)k;
    grec[k] = r; okey[k] = order_key(r);
    if (!valid) fs_raise(v.flag, FS_FLAG_STATE);
  }
}


// ---- scan order of the dense placement kernel --------------------------------------------------
// GPUs that can take a COLD request at all (1 <= n_res < RMAX, sm_free >= 1, co-residents feasible
// at some phi) in ascending order of d_k = a_min_k - Ecur_k, the request-independent part of the
// pruning bound fl(fl(a_min + b) - Ecur); everything else follows as sentinels no request is
// eligible for.  Placement results do not depend on this order (ties compare (dE, k) in full): it
// only decides how soon a request meets its best GPUs and can stop scanning (fs_place.cu).
// rank of every record by (key, index): warp <-> record, lanes over the other records' keys
// (written by the summary kernel), partial counts summed by shuffles
__device__ __forceinline__ void order_rank_block(int bid, const FsGpuRec* __restrict__ grec,
                                                 const float* __restrict__ okey, int Kpad,
                                                 FsGpuRec* __restrict__ gsort, double* __restrict__ dsort) {
  const int lane = threadIdx.x & 31;
  const int i = bid * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (i >= Kpad) return;
  const float key = okey[i];
  int rank = 0;
  for (int j = lane; j < Kpad; j += 32) {
    const float kj = okey[j];
    rank += (kj < key || (kj == key && j < i)) ? 1 : 0;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rank += __shfl_xor_sync(0xffffffffu, rank, o);
  if (lane != 0) return;
  FsGpuRec mine = grec[i];
  double dd = (double)FS_INF;
  if (cold_capable(mine)) { dd = (double)mine.a_min - (double)mine.e_cur; mine.k = (uint32_t)i; }
  else {     // sentinel: mem_free = -INF fails every memory test
    mine.t_avail_ms = 0.f; mine.mem_free_mb = -FS_INF; mine.e_cur = 0.f; mine.meta = 1u | (1u << 8);
    for (int j = 0; j < FS_RMAX; ++j) mine.model[j] = -1;
    mine.a_min = FS_INF; mine.k = 0u;
  }
  gsort[rank] = mine; dsort[rank] = dd;
}
// dsuf[0] = max over the capable GPUs of max(a_min, |Ecur|) (INF if any is huge: no early stop);
// dsuf[1+c] = min of d over sorted positions >= 32*c   (exact suffix minimum, in double);
// dsuf[2+nchunk] = the earliest T_avail among the capable GPUs
__device__ __forceinline__ void order_suffix_block(const FsGpuRec* __restrict__ gsort,
                                                   const double* __restrict__ dsort, int nchunk,
                                                   double* __restrict__ dsuf) {
  __shared__ double seg[1024];
  __shared__ float smax[32], smin[32];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  float amax = 0.0f, tmin = FS_INF;
  for (int c = warp; c < nchunk; c += 32) {            // warp <-> chunk, lane <-> record
    const int pos = c * FS_CHUNK + lane;
    double m = dsort[pos];
    if (m < (double)FS_INF) {
      amax = fmaxf(amax, fmaxf(gsort[pos].a_min, fabsf(gsort[pos].e_cur)));
      tmin = fminf(tmin, gsort[pos].t_avail_ms);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { const double u = __shfl_xor_sync(0xffffffffu, m, o); m = u < m ? u : m; }
    if (lane == 0) dsuf[1 + c] = m;
  }
  __syncthreads();
  const int per = (nchunk + 1023) / 1024;
  const int lo = min(nchunk, t * per), hi = min(nchunk, lo + per);
  double m = (double)FS_INF;
  for (int c = lo; c < hi; ++c) { const double dv = dsuf[1 + c]; m = dv < m ? dv : m; }
  seg[t] = m;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {           // inclusive suffix-minimum scan of the segments
    const double dv = t + off < 1024 ? seg[t + off] : (double)FS_INF;
    __syncthreads();
    if (dv < seg[t]) seg[t] = dv;
    __syncthreads();
  }
  double carry = t + 1 < 1024 ? seg[t + 1] : (double)FS_INF;   // min over the segments after mine
  for (int c = hi - 1; c >= lo; --c) {
    const double dv = dsuf[1 + c];
    carry = dv < carry ? dv : carry;
    dsuf[1 + c] = carry;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    tmin = fminf(tmin, __shfl_xor_sync(0xffffffffu, tmin, o));
  }
  if (lane == 0) { smax[warp] = amax; smin[warp] = tmin; }
  __syncthreads();
  if (t == 0) {
    for (int w = 1; w < 32; ++w) { amax = fmaxf(amax, smax[w]); tmin = fminf(tmin, smin[w]); }
    dsuf[0] = amax <= 1e37f ? (double)amax : (double)FS_INF;
    dsuf[1 + nchunk] = (double)FS_INF;
    dsuf[2 + nchunk] = (double)tmin;                   // earliest T_avail of a cold-capable GPU (NaN-free: min)
  }
}

// ---- warm lists: for every model, the (GPU, tenant slot) pairs that host it -----------------
__device__ __forceinline__ void warm_count_block(int bid, const FsView& v, int32_t* __restrict__ cnt /*[M+1], zeroed*/) {
  const int k = bid * blockDim.x + threadIdx.x;
  if (k >= v.K) return;
  const FsGpuInfo gi = v.ginfo[k];
  for (int i = 0; i < gi.n_res; ++i) {
    bool first = true;   // only the LOWEST slot with this model is the join target
    for (int j = 0; j < i; ++j) first = first && (gi.model[j] != gi.model[i]);
    if (first) atomicAdd(&cnt[gi.model[i] + 1], 1);
  }
}
// The placement preparation in three launches instead of five (each is launch latency, not work):
//   A  blocks [0, nb_rank): rank sort of the scan order;  blocks [nb_rank, ...): count the warm pairs per model
//   B  block 0: suffix minima of the scan order;          block 1: scan of the per-model counts
//   C  fill the per-model lists
__global__ void __launch_bounds__(256) prep_rank_count_kernel(FsView v, int nb_rank, const FsGpuRec* __restrict__ grec,
                                                             const float* __restrict__ okey, FsGpuRec* __restrict__ gsort,
                                                             double* __restrict__ dsort, int32_t* __restrict__ cnt) {
  if ((int)blockIdx.x < nb_rank) order_rank_block((int)blockIdx.x, grec, okey, v.Kpad, gsort, dsort);
  else warm_count_block((int)blockIdx.x - nb_rank, v, cnt);
}
__global__ void __launch_bounds__(1024) prep_suffix_scan_kernel(const FsGpuRec* __restrict__ gsort,
                                                               const double* __restrict__ dsort, int nchunk,
                                                               double* __restrict__ dsuf, int32_t* __restrict__ off,
                                                               int32_t* __restrict__ cursor, int M) {
  if (blockIdx.x == 0) order_suffix_block(gsort, dsort, nchunk, dsuf);
  else fs_bucket_scan_block(off, cursor, M);
}
// one warp per (GPU, slot): lanes over phi reduce the bounds the placement kernel prunes with
__global__ void __launch_bounds__(128) warm_fill_kernel(FsView v, const int32_t* __restrict__ off,
                                                       int32_t* __restrict__ cursor,
                                                       FsWarmItem* __restrict__ items) {
  const int lane = threadIdx.x & 31;
  const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int k = w >> 2, i = w & 3;
  if (k >= v.K) return;
  const FsGpuInfo gi = v.ginfo[k];
  if (i >= gi.n_res) return;
  for (int j = 0; j < i; ++j) if (gi.model[j] == gi.model[i]) return;   // not the join target
  const FsDimsDev d = v.d;
  const int m = gi.model[i], br1 = gi.br1[i];
  float a_min = FS_INF;
  FsPlaneMin pm; pm.lpf = FS_INF; pm.lmin = FS_INF; pm.eta = 0.0f; pm._pad = 0.0f;
  for (int phi = lane; phi < d.F; phi += 32) a_min = fminf(a_min, v.gA[((size_t)k * FS_NVAR + 1 + i) * d.F + phi]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a_min = fminf(a_min, __shfl_xor_sync(0xffffffffu, a_min, o));
  if (br1 >= 0 && gi.sm_free >= 1) {                   // minima over shares < sm_free, all phi: one lookup
    pm = v.pmin[(((size_t)m * 2 + 1) * d.B + br1) * d.S + gi.sm_free - 1];
  }
  if (lane == 0) {
    FsWarmItem it;
    it.k = k; it.j = i; it.br1 = br1; it.sm_free = gi.sm_free;
    it.t_avail_ms = gi.t_avail_ms; it.mem_free_mb = gi.mem_free_mb; it.e_cur = gi.e_cur;
    it.a_min = a_min; it.lp1f = pm.lpf; it.eta1 = pm.eta; it.l1_min = pm.lmin; it._pad0 = 0u; it.f_cur = gi.f_cur;
    it.magic = fs_magic((uint32_t)max(br1, 0) + 1u); it._pad[0] = it._pad[1] = 0;
    items[off[m] + atomicAdd(&cursor[m], 1)] = it;
  }
}

}  // namespace

int fsk_summary(const FsView& v, FsGpuInfo* ginfo, float* gA, FsGpuRec* grec, float* gA0, float* okey,
                cudaStream_t st, FsTimers* tm) {
  if (v.K <= 0) return 0;
  const int wpb = 4;
  fs_tm_beg(tm, FS_T_SUMMARY, st);
  summary_kernel<<<(v.Kpad + wpb - 1) / wpb, wpb * 32, 0, st>>>(v, ginfo, gA, grec, gA0, okey);
  fs_tm_end(tm, FS_T_SUMMARY, st);
  return 1;
}

// What only the placement entry points need (built lazily by their first call after fs_set_gpu_state):
// the scan order of the scoring kernel and the per-model warm lists.
int fsk_place_prepare(const FsView& v, const FsGpuRec* grec, FsGpuRec* gsort, double* dsort, double* dsuf,
                      int32_t* warm_off, int32_t* warm_cursor, FsWarmItem* items, cudaStream_t st, FsTimers* tm) {
  if (v.K <= 0) return 0;
  fs_tm_beg(tm, FS_T_PLACE_WARM, st);
  const float* okey = reinterpret_cast<const float*>(dsuf + v.Kpad / FS_CHUNK + 4);   // written by the summary kernel
  cudaMemsetAsync(warm_off, 0, sizeof(int32_t) * (v.d.M + 1), st);
  const int nb_rank = (v.Kpad + 7) / 8, nb_count = (v.K + 255) / 256;
  prep_rank_count_kernel<<<nb_rank + nb_count, 256, 0, st>>>(v, nb_rank, grec, okey, gsort, dsort, warm_off);
  prep_suffix_scan_kernel<<<2, 1024, 0, st>>>(gsort, dsort, v.Kpad / FS_CHUNK, dsuf, warm_off, warm_cursor, v.d.M);
  warm_fill_kernel<<<(v.K * FS_RMAX + 3) / 4, 128, 0, st>>>(v, warm_off, warm_cursor, items);
  fs_tm_end(tm, FS_T_PLACE_WARM, st);
  return 3;
}
