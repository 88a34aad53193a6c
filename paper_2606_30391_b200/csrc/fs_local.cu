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
                                                        uint32_t flags, float* __restrict__ Gs) {
  const FsDimsDev d = v.d;
  const int gi = blockIdx.x, slot = blockIdx.y, i = slot >> 1, p = slot & 1;
  int k = gpu_ids ? gpu_ids[gi] : gi;
  const int rows = d.F * d.S;
  float* g_out = Gs + ((size_t)gi * (FS_RMAX * 2) + slot) * rows;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  if (k < 0 || k >= v.K) return;                       // flagged by the split kernel
  const int n_res = v.ginfo[k].n_res;                  // 0 if the record was invalid
  if (i >= n_res) return;
  const fs_tenant t = v.states[k].t[i];
  const uint32_t q = t.q[p];
  const bool obj_power = flags & FS_OBJ_POWER;
  if (q == 0) {
    for (int row = threadIdx.x; row < rows; row += blockDim.x) g_out[row] = 0.0f;
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
    if (lane == 0) g_out[row] = key == FS_KEY_NONE ? FS_INF : fs_unorderable((uint32_t)(key >> 32));
  }
}

// ---- step 1, table-major: slots grouped by (model, phase) so that every LUT row is read once ----
// Per call the live slots (q > 0) are counting-sorted by bin = (model*2+phase)*QB + q-bucket.
// A block takes one non-empty (model, phase) key and a tile of LS_TR consecutive (phi,sigma)
// rows, stages their LAT/POW vectors over beta in shared memory (1-D TMA bulk copies; the rows of
// a tile are contiguous in the caller's layout), and its warps walk the key's slots 32 at a
// time: lane <-> slot, sequential over beta, LDS.128 broadcasts of four beta per row, rounds by
// multiply-high with a per-beta magic constant (exact for q < 2^24, beta < 256).  Strict '<' in
// ascending beta keeps the lowest beta on ties, as the definition wants.
constexpr int LS_TR = 16;         // rows per tile (a multiple of 8; 2 x 16 x B floats of shared memory: 32 KB at B = 256)
constexpr int LS_QB = FS_LOCAL_QB; // q buckets per key: slots of (nearly) the same depth share a warp, so its lanes stop together
constexpr int LS_WARPS = 4;
__constant__ uint32_t c_magic[FS_MAX_B];   // ceil(2^32 / (beta+1)), beta >= 1

struct __align__(16) LocalSlot { int32_t gi; uint32_t q; float slo; uint32_t meta; };  // meta = slot | nb << 8

__device__ __forceinline__ bool local_slot_of(const FsView& v, const int32_t* gpu_ids, int gi, int slot,
                                              LocalSlot& o, int& bin) {
  const int k = gpu_ids ? gpu_ids[gi] : gi;
  if (k < 0 || k >= v.K) return false;
  const int i = slot >> 1, p = slot & 1;
  if (i >= v.ginfo[k].n_res) return false;
  const fs_tenant& t = v.states[k].t[i];
  const uint32_t q = t.q[p];
  if (q == 0) return false;
  const uint32_t nb = q < (uint32_t)v.d.B ? q : (uint32_t)v.d.B;
  o.gi = gi; o.q = q; o.slo = t.slo_ms[p]; o.meta = (uint32_t)slot | (nb << 8);
  bin = (t.model * 2 + p) * LS_QB + (int)(((nb - 1) * LS_QB) / (uint32_t)v.d.B);
  return true;
}
__global__ void local_bin_count_kernel(FsView v, int n, const int32_t* __restrict__ gpu_ids, int32_t* __restrict__ off) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x >= n * FS_RMAX * 2) return;
  LocalSlot o; int bin;
  if (local_slot_of(v, gpu_ids, x >> 3, x & 7, o, bin)) atomicAdd(&off[bin + 1], 1);
}
__global__ void local_bin_fill_kernel(FsView v, int n, const int32_t* __restrict__ gpu_ids,
                                      const int32_t* __restrict__ off, int32_t* __restrict__ cursor,
                                      LocalSlot* __restrict__ slots) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x >= n * FS_RMAX * 2) return;
  LocalSlot o; int bin;
  if (local_slot_of(v, gpu_ids, x >> 3, x & 7, o, bin)) slots[off[bin] + atomicAdd(&cursor[bin], 1)] = o;
}
// one block: the scan of the bin counts, then the list of the non-empty (model, phase) keys (one launch, not two)
__global__ void __launch_bounds__(1024) local_scan_keys_kernel(int32_t* __restrict__ off, int32_t* __restrict__ cursor, int nbins,
                                                              int nkeys_all, int32_t* __restrict__ keylist,
                                                              int32_t* __restrict__ nkeys) {
  fs_bucket_scan_block(off, cursor, nbins);
  __syncthreads();
  for (int key = threadIdx.x; key < nkeys_all; key += blockDim.x)
    if (off[(key + 1) * LS_QB] > off[key * LS_QB]) keylist[atomicAdd(nkeys, 1)] = key;
}

// the body for one phase (P = key & 1): the deadline rule differs (prefill: whole queue; decode: one step), so the
// candidate loop is compiled once per phase and the block picks its version once
template <int P, bool OBJ_POWER, bool fill>
__device__ __forceinline__ void local_slot_body(const FsView& v, const int key, unsigned char* ls_smem, uint64_t& bar,
                                                const int32_t* __restrict__ off,
                                                const LocalSlot* __restrict__ slots, float* __restrict__ Gs) {
  const FsDimsDev d = v.d;
  const int B = d.B, rows = d.F * d.S;
  const int r0 = blockIdx.y * LS_TR, tr = min(LS_TR, rows - r0);
  float* sl = reinterpret_cast<float*>(ls_smem);            // [LS_TR][B]
  float* sp = sl + LS_TR * B;                               // [LS_TR][B]
  const size_t src = ((size_t)key * rows + r0) * B;
  const uint32_t bytes = (uint32_t)tr * B * sizeof(float);
  if (threadIdx.x == 0) { fs_mbar_init(&bar, 1); fs_mbar_fence_init(); }
  __syncthreads();
  if (threadIdx.x == 0) {
    fs_mbar_expect_tx(&bar, 2 * bytes);
    fs_tma_load_1d(sl, v.lat + src, bytes, &bar);
    fs_tma_load_1d(sp, v.pow + src, bytes, &bar);
  }
  if (tr < LS_TR)   // ragged last tile: keep the unused rows finite
    for (int x = threadIdx.x + tr * B; x < LS_TR * B; x += blockDim.x) { sl[x] = 1.0f; sp[x] = 1.0f; }
  fs_mbar_wait(&bar, 0);
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int s0 = off[key * LS_QB], s1 = off[(key + 1) * LS_QB];
  // Rounds of LS_WARPS*32 slots, lane <-> slot.  In a round that is not full the slots fill whole warps first
  // (every lane busy) and the remaining r < 32 slots go to one more warp, where each slot gets G = 32 / r
  // lanes (at most 8) that split the beta range (groups of four beta, interleaved; their minima are merged by
  // shuffles: min is exact in any order): a warp left with 4 slots finishes 8 times sooner instead of running 4
  // lanes over the whole range (4,096 GPUs: 0.761 -> 0.717 ms).  With `fill` = false (the per-phase launches used for grids
  // of a few waves) only a round of fewer than 64 slots is split, and it is spread EVENLY over the block's warps,
  // so that every warp works and the block is short (pod, ~40 slots per key: 0.185 against 0.194 - 0.213 ms).
  for (int start = s0; start < s1; start += LS_WARPS * 32) {
    const int n_round = min(LS_WARPS * 32, s1 - start);
    int per = 32, base = warp * 32;                     // slots of this warp, and where they start in the round
    if (!fill) {
      if (n_round < 64) { per = (n_round + LS_WARPS - 1) / LS_WARPS; base = warp * per; }
    } else if (n_round < LS_WARPS * 32) {
      const int nfull = n_round >> 5, rem = n_round & 31;
      per = warp < nfull ? 32 : (warp == nfull ? rem : 0);
    }
    // a warp with fewer than 17 slots gives each slot G lanes (any G up to 8, not only powers of two: 10 slots
    // -> 3 groups of 10 lanes) that split the beta range; lanes beyond G * per idle
    const int G = per > 0 ? min(32 / per, 8) : 1;
    const int grp = per > 0 ? lane / per : 0, idx = per > 0 ? lane - grp * per : lane, sl_ix = base + idx;
    const bool have = per > 0 && grp < G && sl_ix < n_round;
    LocalSlot sl_ = have ? slots[start + sl_ix] : LocalSlot{0, 0u, 0.f, 0u};
    const uint32_t nb = have ? (sl_.meta >> 8) : 0u;
    uint32_t maxnb;
    asm volatile("redux.sync.max.u32 %0, %1, 0xffffffff;" : "=r"(maxnb) : "r"(nb));
    float best[LS_TR];
#pragma unroll
    for (int r = 0; r < LS_TR; ++r) best[r] = FS_INF;
    for (uint32_t b4 = 4u * grp; b4 < maxnb; b4 += 4u * G) {
      // the four betas' round counts and deadlines once per lane and trip, shared by all rows of the tile
      float fr[4], slo_b[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const uint32_t beta = b4 + u;
        const uint32_t rounds = beta == 0 ? sl_.q : __umulhi(sl_.q + beta, c_magic[beta]);
        fr[u] = __uint2float_rn(rounds);
        // beta past this slot's range: a deadline nothing meets (tables are > 0)
        slo_b[u] = beta < nb ? sl_.slo : -1.0f;
      }
#pragma unroll
      for (int rh = 0; rh < LS_TR; rh += 8) {          // eight rows at a time: 16 broadcast LDS.128 in flight
        float4 L4[8], P4[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          L4[r] = *reinterpret_cast<const float4*>(sl + (rh + r) * B + b4);
          P4[r] = *reinterpret_cast<const float4*>(sp + (rh + r) * B + b4);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
          for (int r = 0; r < 8; ++r) {
            const float la = u == 0 ? L4[r].x : u == 1 ? L4[r].y : u == 2 ? L4[r].z : L4[r].w;
            const float pw = u == 0 ? P4[r].x : u == 1 ? P4[r].y : u == 2 ? P4[r].z : P4[r].w;
            const float t = __fmul_rn(fr[u], la);
            const float cost = OBJ_POWER ? pw : __fmul_rn(t, pw);
            // one compare + one predicated min per candidate (the ALU pipe binds this kernel);
            // beta* is recovered for the chosen row only (split kernel)
            asm("{.reg .pred p; setp.le.f32 p, %1, %2; @p min.f32 %0, %0, %3;}"
                : "+f"(best[rh + r]) : "f"(P == 0 ? t : la), "f"(slo_b[u]), "f"(cost));
          }
        }
      }
    }
    for (int g = 1; g < G; ++g) {                        // group 0 collects the groups' minima
#pragma unroll
      for (int r = 0; r < LS_TR; ++r) best[r] = fminf(best[r], __shfl_sync(0xffffffffu, best[r], (idx + g * per) & 31));
    }
    if (have && grp == 0) {
      const size_t o = ((size_t)sl_.gi * (FS_RMAX * 2) + (sl_.meta & 0xFF)) * rows + r0;
      if (tr == LS_TR && (rows & 3) == 0) {
#pragma unroll
        for (int r = 0; r < LS_TR; r += 4)
          *reinterpret_cast<float4*>(Gs + o + r) = make_float4(best[r], best[r + 1], best[r + 2], best[r + 3]);
      } else {
#pragma unroll
        for (int r = 0; r < LS_TR; ++r) if (r < tr) Gs[o + r] = best[r];
      }
    }
  }
}

// PSEL = 0 / 1: one launch per phase (the block returns when its key belongs to the other one; the prefill version
// needs fewer registers, which is what matters when a launch is a wave or two: 1,024 GPUs 0.182 against 0.184 ms).
// PSEL = -1: one launch for both phases, every block of the grid has work and no launch waits for the other's tail
// (4,096 GPUs: 0.847 -> 0.785 ms).
template <bool OBJ_POWER, int PSEL>
__global__ void __launch_bounds__(LS_WARPS * 32) local_slot_grouped_kernel(
    FsView v, const int32_t* __restrict__ off, const int32_t* __restrict__ keylist,
    const int32_t* __restrict__ nkeys, const LocalSlot* __restrict__ slots, float* __restrict__ Gs) {
  extern __shared__ __align__(128) unsigned char ls_smem[];
  __shared__ __align__(8) uint64_t bar;
  if ((int)blockIdx.x >= *nkeys) return;
  const int key = keylist[blockIdx.x];
  if (PSEL >= 0) {
    if ((key & 1) != PSEL) return;
    local_slot_body<(PSEL > 0 ? 1 : 0), OBJ_POWER, false>(v, key, ls_smem, bar, off, slots, Gs);
  } else if (key & 1) local_slot_body<1, OBJ_POWER, true>(v, key, ls_smem, bar, off, slots, Gs);
  else                local_slot_body<0, OBJ_POWER, true>(v, key, ls_smem, bar, off, slots, Gs);
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

__global__ void __launch_bounds__(512) local_split_kernel(FsView v, int n,
                                                         const int32_t* __restrict__ gpu_ids,
                                                         uint32_t flags,
                                                         const float* __restrict__ Gs,
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
  for (int i = 0; i < n_res; ++i) {
    // a slot with an empty queue costs 0 (the slot kernels do not visit it)
    const bool q0 = v.states[k].t[i].q[0] != 0, q1 = v.states[k].t[i].q[1] != 0;
    const float* ga = g_in + (size_t)(i * 2) * rows; const float* gb = ga + rows;
    for (int row = threadIdx.x; row < rows; row += blockDim.x)
      sG[i * rows + row] = __fadd_rn(q0 ? ga[row] : 0.0f, q1 ? gb[row] : 0.0f);
  }
  __syncthreads();
  const bool minsm = flags & FS_SPLIT_MINSM;
  unsigned long long key = FS_KEY_NONE;
  uint32_t fphi = 0xFFFFFFFFu;
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
        fphi = min(fphi, (uint32_t)phi);
      }
    }
  } else {
    const uint32_t* cp = comp + (size_t)(n_res - 1) * ns_stride;
    // thread <-> split (rank), inner loop over phi: no division per candidate, the four shared-memory
    // offsets of a split are formed once; (cost, flat) compared in full because flat = phi*NS + rank is
    // not visited in ascending order
    float bestC = FS_INF; uint32_t bflat = 0xFFFFFFFFu;
    // few splits (1 / 15 / 105 for 1-3 tenants): PG thread groups share them and divide the frequencies
    const uint32_t PG = NS >= blockDim.x ? 1u : min((uint32_t)d.F, blockDim.x / NS);
    const uint32_t pg = PG > 1 ? threadIdx.x / NS : 0u;
    for (uint32_t rank = PG > 1 ? threadIdx.x % NS : threadIdx.x; rank < NS && pg < PG; rank += PG > 1 ? NS : blockDim.x) {
      const uint32_t pk = cp[rank];
      int off[FS_RMAX];
#pragma unroll
      for (int i = 0; i < FS_RMAX; ++i) off[i] = (i < n_res ? i : 0) * rows + (int)((pk >> (8 * i)) & 0xFF);
      for (int phi = (int)pg; phi < d.F; phi += (int)PG) {
        float C = sG[off[0] + phi * d.S];
#pragma unroll
        for (int i = 1; i < FS_RMAX; ++i) if (i < n_res) C = __fadd_rn(C, sG[off[i] + phi * d.S]);
        const uint32_t flat = (uint32_t)phi * NS + rank;
        if (C < FS_INF) {
          if (C < bestC || (C == bestC && flat < bflat)) { bestC = C; bflat = flat; }
          fphi = min(fphi, (uint32_t)phi);
        }
      }
    }
    if (bflat != 0xFFFFFFFFu) key = fs_make_key(bestC, bflat);
  }
  // f_req = lowest phi with any feasible candidate: tracked beside the key, reduced as a key of its own
  unsigned long long fkey = fphi == 0xFFFFFFFFu ? FS_KEY_NONE : (unsigned long long)fphi;
  key = block_min_key(key, sred);
  fkey = block_min_key(fkey, sred);
  // ---- outputs.  The slot kernels keep only the minimum cost per (slot, phi, sigma); the batch
  // bucket beta* = lowest beta attaining it is recovered here, for the CHOSEN row of each slot only:
  // warp <-> slot, lanes over beta, first feasible beta whose cost equals the stored minimum.
  __shared__ int sbeta[FS_RMAX * 2];
  uint32_t pk = 0; int phi = -1;
  if (key != FS_KEY_NONE) {
    const uint32_t flat = (uint32_t)key;
    phi = minsm ? (int)flat : (int)(flat / NS);
    if (minsm) {
      for (int i = 0; i < n_res; ++i)
        for (int s = 0; s < d.S; ++s) if (sG[i * rows + phi * d.S + s] < FS_INF) { pk |= (uint32_t)s << (8 * i); break; }
    } else pk = comp[(size_t)(n_res - 1) * ns_stride + flat % NS];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31, i = w >> 1, p = w & 1;
    if (w < FS_RMAX * 2) {
      int bstar = 0;
      const uint32_t q = i < n_res ? v.states[k].t[i].q[p] : 0u;
      if (q > 0) {
        const fs_tenant& tt = v.states[k].t[i];
        const int sg = (pk >> (8 * i)) & 0xFF;
        const float target = g_in[(size_t)(i * 2 + p) * rows + phi * d.S + sg], slo = tt.slo_ms[p];
        const size_t base = fs_idx(d, tt.model, p, phi, sg, 0);
        const int nb = (int)(q < (uint32_t)d.B ? q : (uint32_t)d.B);
        const bool obj_power = flags & FS_OBJ_POWER;
        bstar = -1;
        for (int b0 = 0; b0 < nb && bstar < 0; b0 += 32) {
          const int beta = b0 + lane;
          bool hit = false;
          if (beta < nb) {
            const float la = v.lat[base + beta], pw = v.pow[base + beta];
            const float t = __fmul_rn(__uint2float_rn(fs_ceil_div(q, (uint32_t)beta + 1u)), la);
            const bool ok = p == 0 ? (t <= slo) : (la <= slo);
            hit = ok && (obj_power ? pw : __fmul_rn(t, pw)) == target;
          }
          const unsigned m = __ballot_sync(0xffffffffu, hit);
          if (m) bstar = b0 + __ffs(m) - 1;
        }
        if (bstar < 0) bstar = 0;
      }
      if (lane == 0) sbeta[w] = bstar;
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (key != FS_KEY_NONE) {
      o.phi = (int16_t)phi; o.f_req = (int16_t)(int)fkey; o.flat = (uint32_t)key;
      o.cost = fs_unorderable((uint32_t)(key >> 32));
      const fs_gpu_state& g = v.states[k];
      float E = 0.0f, PW = 0.0f;
      for (int i = 0; i < n_res; ++i) {
        const int sg = (pk >> (8 * i)) & 0xFF;
        o.sigma[i] = (uint8_t)sg;
        float e[2], pw[2];
        for (int p = 0; p < 2; ++p) {
          const uint32_t q = g.t[i].q[p];
          const int beta = q ? sbeta[i * 2 + p] : 0;
          o.beta[i][p] = (uint8_t)beta;
          e[p] = 0.0f; pw[p] = 0.0f;
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
  uint32_t magic[FS_MAX_B];
  magic[0] = 0xFFFFFFFFu;   // unused (beta == 0: rounds = q)
  for (uint32_t n = 2; n <= FS_MAX_B; ++n) magic[n - 1] = (uint32_t)(((1ull << 32) + n - 1) / n);
  int e = (int)cudaMemcpyToSymbol(c_magic, magic, sizeof(magic));
  // [RMAX][F][S] floats at the largest supported dims = 128 KiB
  e |= (int)cudaFuncSetAttribute(local_split_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)(sizeof(float) * FS_RMAX * FS_MAX_F * FS_MAX_S));
  return e;
}

int fsk_local(const FsView& v, int n, const int32_t* gpu_ids, uint32_t flags, fs_local_cfg* out,
              const FsLocalScratch& sc, cudaStream_t st, FsTimers* tm) {
  if (n <= 0) return 0;
  const int rows = v.d.F * v.d.S;
  int launches = 0;
  fs_tm_beg(tm, FS_T_LOCAL_SLOT, st);
  if (v.d.B % 4 == 0) {
    const int nkeys_all = v.d.M * 2, nbins = nkeys_all * LS_QB, nslots = n * FS_RMAX * 2;
    cudaMemsetAsync(sc.bin_off, 0, sizeof(int32_t) * (size_t)(nbins + 1), st);
    cudaMemsetAsync(sc.nkeys, 0, sizeof(int32_t), st);
    local_bin_count_kernel<<<(nslots + 255) / 256, 256, 0, st>>>(v, n, gpu_ids, sc.bin_off);
    local_scan_keys_kernel<<<1, 1024, 0, st>>>(sc.bin_off, sc.bin_cursor, nbins, nkeys_all, sc.keylist, sc.nkeys);
    local_bin_fill_kernel<<<(nslots + 255) / 256, 256, 0, st>>>(v, n, gpu_ids, sc.bin_off, sc.bin_cursor,
                                                               reinterpret_cast<LocalSlot*>(sc.slots));
    const dim3 grid(min(nkeys_all, nslots), (rows + LS_TR - 1) / LS_TR);
    const size_t smem = sizeof(float) * 2 * LS_TR * v.d.B;
    const LocalSlot* sl = reinterpret_cast<const LocalSlot*>(sc.slots);
#define FS_LAUNCH_SLOT(OBJ, PS) \
  local_slot_grouped_kernel<OBJ, PS><<<grid, LS_WARPS * 32, smem, st>>>(v, sc.bin_off, sc.keylist, sc.nkeys, sl, sc.G)
    const bool power = flags & FS_OBJ_POWER;
    if (n >= 2048) {
      if (power) FS_LAUNCH_SLOT(true, -1); else FS_LAUNCH_SLOT(false, -1);
      launches += 4;
    } else {
      if (power) { FS_LAUNCH_SLOT(true, 0); FS_LAUNCH_SLOT(true, 1); } else { FS_LAUNCH_SLOT(false, 0); FS_LAUNCH_SLOT(false, 1); }
      launches += 5;
    }
#undef FS_LAUNCH_SLOT
  } else {
    local_slot_kernel<<<dim3(n, FS_RMAX * 2), 256, 0, st>>>(v, n, gpu_ids, flags, sc.G);
    launches += 1;
  }
  fs_tm_end(tm, FS_T_LOCAL_SLOT, st);
  const size_t smem = sizeof(float) * FS_RMAX * rows;
  fs_tm_beg(tm, FS_T_LOCAL_SPLIT, st);
  // one block per GPU; with several waves of blocks the smaller block fills the SMs more evenly (measured: 4,096
  // GPUs 0.141 -> 0.124 ms with 256 threads, 1,024 GPUs 0.046 -> 0.049 ms)
  local_split_kernel<<<n, n >= 2048 ? 256 : 512, smem, st>>>(v, n, gpu_ids, flags, sc.G, sc.comp, sc.comp_n,
                                           sc.ns_stride, out);
  fs_tm_end(tm, FS_T_LOCAL_SPLIT, st);
  return launches + 1;
}
