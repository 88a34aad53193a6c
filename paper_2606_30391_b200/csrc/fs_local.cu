// fs_local.cu — fs_local_config: per-GPU runtime resource allocation (§3.4, Fig. 8
// step 3 P:206-210): frequency sweep, per-task SM allocation, lowest predicted energy
// or power (R:s8); batching as one batch bucket per slot (R:s10).
//
// Hierarchical definition:
//   1. slot (i,p) at (phi,sigma): g = min over beta < min(B,q), deadline ok, of the slot cost;
//      beta* = lowest beta attaining it; q == 0 -> cost 0, beta* 0.
//   2. tenant: G_i[phi][sigma] = fl(g_i0 + g_i1)
//   3. EXHAUSTIVE: min over phi x compositions (sum(sigma_i+1) == S) of the slot-order sum,
//      flat = phi*NS + lexicographic rank;   MINSM: per phi the lowest feasible sigma per
//      tenant, sum <= S (Fig. 8 accepts exactly 100 %, R:s7), flat = phi.
#include "fs_kernels.h"

namespace {

// ---- step 1: batch search of one slot row, one warp per (phi,sigma) row, lanes over beta ----
// grid = (n GPUs, RMAX*2 slots); rows strided over the block's warps.
__global__ void __launch_bounds__(256) local_slot_kernel(FsView v, int n,
                                                        const int32_t* __restrict__ gpu_ids,
                                                        uint32_t flags, float* __restrict__ Gs,
                                                        uint8_t* __restrict__ Bs) {
  const FsDimsDev d = v.d;
  const int gi = blockIdx.x, slot = blockIdx.y, i = slot >> 1, p = slot & 1;
  int k = gpu_ids ? gpu_ids[gi] : gi;
  const int rows = d.F * d.S;
  float* g_out = Gs + ((size_t)gi * (FS_RMAX * 2) + slot) * rows;
  uint8_t* b_out = Bs + ((size_t)gi * (FS_RMAX * 2) + slot) * rows;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  if (k < 0 || k >= v.K) return;                       // flagged by the split kernel
  const int n_res = v.ginfo[k].n_res;                  // 0 if the record was invalid
  if (i >= n_res) return;
  const fs_tenant t = v.states[k].t[i];
  const uint32_t q = t.q[p];
  const bool obj_power = flags & FS_OBJ_POWER;
  if (q == 0) {
    for (int row = threadIdx.x; row < rows; row += blockDim.x) { g_out[row] = 0.0f; b_out[row] = 0; }
    return;
  }
  const float slo = t.slo_ms[p];
  const int nb = (int)(q < (uint32_t)d.B ? q : (uint32_t)d.B);
  for (int row = warp; row < rows; row += nwarp) {     // row = phi*S + sigma (logical layout)
    const size_t base = (((size_t)t.model * 2 + p) * rows + row) * d.B;
    unsigned long long key = FS_KEY_NONE;
    for (int beta = lane; beta < nb; beta += 32) {
      const float lat = v.lat[base + beta], pw = v.pow[base + beta];
      const FsSlot s = fs_slot(p, lat, pw, fs_ceil_div(q, (uint32_t)beta + 1u), 0.0f, slo);
      const float cost = obj_power ? pw : s.e;
      if (s.ok && cost < FS_INF) {
        const unsigned long long kk = fs_make_key(cost, (uint32_t)beta);
        key = kk < key ? kk : key;
      }
    }
    key = fs_warp_min_key(key);
    if (lane == 0) {
      g_out[row] = key == FS_KEY_NONE ? FS_INF : fs_unorderable((uint32_t)(key >> 32));
      b_out[row] = key == FS_KEY_NONE ? 0 : (uint8_t)(uint32_t)key;
    }
  }
}

// ---- steps 2-3: tenant sums, split search, argmin; one block per GPU -----------------------
__device__ __forceinline__ unsigned long long block_min_key(unsigned long long key,
                                                            unsigned long long* sred) {
  key = fs_warp_min_key(key);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  __syncthreads();
  if (lane == 0) sred[warp] = key;
  __syncthreads();
  if (warp == 0) {
    unsigned long long k2 = lane < nwarp ? sred[lane] : FS_KEY_NONE;
    k2 = fs_warp_min_key(k2);
    if (lane == 0) sred[0] = k2;
  }
  __syncthreads();
  return sred[0];
}

__global__ void __launch_bounds__(256) local_split_kernel(FsView v, int n,
                                                         const int32_t* __restrict__ gpu_ids,
                                                         uint32_t flags,
                                                         const float* __restrict__ Gs,
                                                         const uint8_t* __restrict__ Bs,
                                                         const uint32_t* __restrict__ comp,   // [RMAX][NSmax] packed splits
                                                         const uint32_t* __restrict__ comp_n, // [RMAX] NS per n_res
                                                         int ns_stride,
                                                         fs_local_cfg* __restrict__ out) {
  extern __shared__ float sG[];            // [n_res][F][S] tenant costs
  __shared__ unsigned long long sred[32];
  const FsDimsDev d = v.d;
  const int gi = blockIdx.x;
  const int k = gpu_ids ? gpu_ids[gi] : gi;
  const int rows = d.F * d.S;
  const bool bad_id = (k < 0 || k >= v.K);
  const int n_res = bad_id ? 0 : v.ginfo[k].n_res;
  fs_local_cfg o;
  {
    uint32_t* w = reinterpret_cast<uint32_t*>(&o);
#pragma unroll
    for (int x = 0; x < (int)(sizeof(o) / 4); ++x) w[x] = 0;
  }
  o.phi = -1; o.f_req = -1; o.flat = 0xFFFFFFFFu;
  if (n_res < 1) {                          // inactive GPU: cost 0
    if (threadIdx.x == 0) { out[gi] = o; if (bad_id) fs_raise(v.flag, FS_FLAG_ARG); }
    return;
  }
  o.cost = o.energy_mj = o.power_w = FS_INF;
  if (n_res > d.S) { if (threadIdx.x == 0) out[gi] = o; return; }
  const float* g_in = Gs + (size_t)gi * (FS_RMAX * 2) * rows;
  for (int x = threadIdx.x; x < n_res * rows; x += blockDim.x) {
    const int i = x / rows, row = x % rows;
    sG[x] = __fadd_rn(g_in[(size_t)(i * 2) * rows + row], g_in[(size_t)(i * 2 + 1) * rows + row]);
  }
  __syncthreads();
  const bool minsm = flags & FS_SPLIT_MINSM;
  unsigned long long key = FS_KEY_NONE;
  const uint32_t NS = minsm ? 1u : comp_n[n_res - 1];
  if (minsm) {
    for (int phi = threadIdx.x; phi < d.F; phi += blockDim.x) {
      int tot = 0; bool all = true; float C = 0.0f;
      for (int i = 0; i < n_res; ++i) {
        int sg = -1;
        for (int s = 0; s < d.S; ++s) if (sG[i * rows + phi * d.S + s] < FS_INF) { sg = s; break; }
        if (sg < 0) { all = false; break; }
        tot += sg + 1;
        const float g = sG[i * rows + phi * d.S + sg];
        C = (i == 0) ? g : __fadd_rn(C, g);
      }
      if (all && tot <= d.S && C < FS_INF) {
        const unsigned long long kk = fs_make_key(C, (uint32_t)phi);
        key = kk < key ? kk : key;
      }
    }
  } else {
    const uint32_t* cp = comp + (size_t)(n_res - 1) * ns_stride;
    const uint32_t total = (uint32_t)d.F * NS;
    for (uint32_t c = threadIdx.x; c < total; c += blockDim.x) {
      const uint32_t phi = c / NS, rank = c % NS;
      const uint32_t pk = cp[rank];
      float C = 0.0f;
      for (int i = 0; i < n_res; ++i) {
        const float g = sG[i * rows + phi * d.S + ((pk >> (8 * i)) & 0xFF)];
        C = (i == 0) ? g : __fadd_rn(C, g);
      }
      if (C < FS_INF) {
        const unsigned long long kk = fs_make_key(C, c);
        key = kk < key ? kk : key;
      }
    }
  }
  // f_req = lowest phi with any feasible candidate: min over the low word / NS of feasible keys
  // is not the key minimum, so reduce it separately as a key with value 0.
  unsigned long long fkey = FS_KEY_NONE;
  if (minsm) {
    // feasible phis were exactly those that produced a key; recompute cheaply per thread
    for (int phi = threadIdx.x; phi < d.F; phi += blockDim.x) {
      int tot = 0; bool all = true; float C = 0.0f;
      for (int i = 0; i < n_res; ++i) {
        int sg = -1;
        for (int s = 0; s < d.S; ++s) if (sG[i * rows + phi * d.S + s] < FS_INF) { sg = s; break; }
        if (sg < 0) { all = false; break; }
        tot += sg + 1;
        const float g = sG[i * rows + phi * d.S + sg];
        C = (i == 0) ? g : __fadd_rn(C, g);
      }
      if (all && tot <= d.S && C < FS_INF) { fkey = (unsigned long long)phi; break; }
    }
  } else {
    const uint32_t* cp = comp + (size_t)(n_res - 1) * ns_stride;
    for (int phi = 0; phi < d.F && fkey == FS_KEY_NONE; ++phi) {
      // all threads scan the splits of this phi together
      bool any = false;
      for (uint32_t rank = threadIdx.x; rank < NS && !any; rank += blockDim.x) {
        const uint32_t pk = cp[rank];
        float C = 0.0f;
        for (int i = 0; i < n_res; ++i) {
          const float g = sG[i * rows + phi * d.S + ((pk >> (8 * i)) & 0xFF)];
          C = (i == 0) ? g : __fadd_rn(C, g);
        }
        any = C < FS_INF;
      }
      if (__syncthreads_or(any)) fkey = (unsigned long long)phi;
    }
  }
  key = block_min_key(key, sred);
  fkey = block_min_key(fkey, sred);
  if (threadIdx.x == 0) {
    if (key != FS_KEY_NONE) {
      const uint32_t flat = (uint32_t)key;
      const int phi = minsm ? (int)flat : (int)(flat / NS);
      o.phi = (int16_t)phi; o.f_req = (int16_t)(int)fkey; o.flat = flat;
      o.cost = fs_unorderable((uint32_t)(key >> 32));
      uint32_t pk = 0;
      if (minsm) {
        for (int i = 0; i < n_res; ++i)
          for (int s = 0; s < d.S; ++s) if (sG[i * rows + phi * d.S + s] < FS_INF) { pk |= (uint32_t)s << (8 * i); break; }
      } else pk = comp[(size_t)(n_res - 1) * ns_stride + flat % NS];
      const uint8_t* b_in = Bs + (size_t)gi * (FS_RMAX * 2) * rows;
      const fs_gpu_state& g = v.states[k];
      float E = 0.0f, PW = 0.0f;
      for (int i = 0; i < n_res; ++i) {
        const int sg = (pk >> (8 * i)) & 0xFF;
        o.sigma[i] = (uint8_t)sg;
        float e[2], pw[2];
        for (int p = 0; p < 2; ++p) {
          const int beta = b_in[(size_t)(i * 2 + p) * rows + phi * d.S + sg];
          o.beta[i][p] = (uint8_t)beta;
          e[p] = 0.0f; pw[p] = 0.0f;
          const uint32_t q = g.t[i].q[p];
          if (q > 0) {
            const size_t ix = fs_idx(d, g.t[i].model, p, phi, sg, beta);
            pw[p] = v.pow[ix];
            e[p] = __fmul_rn(__fmul_rn(__uint2float_rn(fs_ceil_div(q, (uint32_t)beta + 1u)), v.lat[ix]), pw[p]);
          }
        }
        const float ei = __fadd_rn(e[0], e[1]), pi = __fadd_rn(pw[0], pw[1]);
        E = (i == 0) ? ei : __fadd_rn(E, ei);
        PW = (i == 0) ? pi : __fadd_rn(PW, pi);
      }
      o.energy_mj = E; o.power_w = PW;
    }
    out[gi] = o;
  }
}

}  // namespace

int fsk_local_smem_attr() {
  // [RMAX][F][S] floats at the largest supported dims = 128 KiB
  return (int)cudaFuncSetAttribute(local_split_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)(sizeof(float) * FS_RMAX * FS_MAX_F * FS_MAX_S));
}

int fsk_local(const FsView& v, int n, const int32_t* gpu_ids, uint32_t flags, fs_local_cfg* out,
              const FsLocalScratch& sc, cudaStream_t st, FsTimers* tm) {
  if (n <= 0) return 0;
  const int rows = v.d.F * v.d.S;
  fs_tm_beg(tm, FS_T_LOCAL_SLOT, st);
  local_slot_kernel<<<dim3(n, FS_RMAX * 2), 256, 0, st>>>(v, n, gpu_ids, flags, sc.G, sc.B);
  fs_tm_end(tm, FS_T_LOCAL_SLOT, st);
  const size_t smem = sizeof(float) * FS_RMAX * rows;
  fs_tm_beg(tm, FS_T_LOCAL_SPLIT, st);
  local_split_kernel<<<n, 256, smem, st>>>(v, n, gpu_ids, flags, sc.G, sc.B, sc.comp, sc.comp_n,
                                           sc.ns_stride, out);
  fs_tm_end(tm, FS_T_LOCAL_SPLIT, st);
  return 2;
}
