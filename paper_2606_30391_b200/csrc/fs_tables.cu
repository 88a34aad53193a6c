// fs_tables.cu — fs_load_profiles device work: validate the LUT and build the
// plane layout [M][2][B][S][F] of {LAT, POW} pairs in which the (sigma,phi) plane of one (model,
// phase, batch bucket) is one contiguous S*F*8-byte block (what placement stages per request with
// one TMA bulk copy), and the per-plane prefix minima the placement bounds are made of.
#include "fs_kernels.h"

namespace {

// One block transposes a 32x32 (phi, beta) tile of one (model, phase, sigma) slice for both
// tables.  Reads are coalesced along beta, writes along phi.
__global__ void __launch_bounds__(256) build_planes_kernel(const float* __restrict__ lat,
                                                          const float* __restrict__ pow,
                                                          float2* __restrict__ lpT, FsDimsDev d,
                                                          int* flag) {
  __shared__ float tl[32][33];
  __shared__ float tp[32][33];
  const int tilesB = (d.B + 31) / 32, tilesF = (d.F + 31) / 32;
  int bid = blockIdx.x;
  const int tb = bid % tilesB; bid /= tilesB;
  const int tf = bid % tilesF; bid /= tilesF;
  const int s = bid % d.S;     bid /= d.S;
  const int mp = bid;  // m*2+p
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
  bool bad = false;
  for (int r = ty; r < 32; r += 8) {
    const int f = tf * 32 + r, b = tb * 32 + tx;
    if (f < d.F && b < d.B) {
      const size_t i = (((size_t)mp * d.F + f) * d.S + s) * d.B + b;
      const float l = lat[i], p = pow[i];
      // every entry finite and > 0 (include/festina_eval.h)
      if (!(l > 0.0f && l < FS_INF && p > 0.0f && p < FS_INF)) bad = true;
      tl[r][tx] = l;
      tp[r][tx] = p;
    }
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int b = tb * 32 + r, f = tf * 32 + tx;
    if (f < d.F && b < d.B) {
      const size_t o = (((size_t)mp * d.B + b) * d.S + s) * d.F + f;
      lpT[o] = make_float2(tl[tx][r], tp[tx][r]);
    }
  }
  if (bad) fs_raise(flag, FS_FLAG_TABLE);
}

// pmin[m][p][b][s] over the plane (m, p, b), shares <= s and all phi: the minimum of the exact product
// LAT*POW (binary64 holds the product of two binary32 values exactly) shrunk by 2^-22 and rounded down, the
// minimum LAT, and 2^-149 (max POW + 1) rounded up.  fs_energy_lb (fs_common.cuh) turns them into a lower
// bound on fl(fl(rounds*LAT)*POW) of every such entry with two binary32 operations.
__global__ void __launch_bounds__(128) plane_min_kernel(const float2* __restrict__ lpT, FsDimsDev d,
                                                       FsPlaneMin* __restrict__ pmin) {
  const int lane = threadIdx.x & 31;
  const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);     // (m*2+p)*B + b
  if (w >= d.M * 2 * d.B) return;
  const float2* pl = lpT + (size_t)w * d.S * d.F;
  double mlp = (double)FS_INF; float ml = FS_INF, xp = 0.0f;
  for (int s = 0; s < d.S; ++s) {
    double lp = (double)FS_INF; float l = FS_INF, p = 0.0f;
    for (int phi = lane; phi < d.F; phi += 32) {
      const float2 e = pl[s * d.F + phi];
      const double pr = (double)e.x * (double)e.y;
      lp = pr < lp ? pr : lp; l = fminf(l, e.x); p = fmaxf(p, e.y);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double u = __shfl_xor_sync(0xffffffffu, lp, o); lp = u < lp ? u : lp;
      l = fminf(l, __shfl_xor_sync(0xffffffffu, l, o)); p = fmaxf(p, __shfl_xor_sync(0xffffffffu, p, o));
    }
    mlp = lp < mlp ? lp : mlp; ml = fminf(ml, l); xp = fmaxf(xp, p);
    if (lane == 0) {
      FsPlaneMin o;
      o.lpf = __double2float_rd(mlp * (1.0 - 0x1p-22)); o.lmin = ml;
      o.eta = __double2float_ru(0x1p-149 * ((double)xp + 1.0)); o._pad = 0.0f;
      pmin[(size_t)w * d.S + s] = o;
    }
  }
}

}  // namespace

int fsk_build_planes(const float* lat, const float* pow, float2* lpT, FsPlaneMin* pmin, FsDimsDev d,
                     int* flag, cudaStream_t st) {
  const long long blocks = (long long)d.M * 2 * d.S * ((d.F + 31) / 32) * ((d.B + 31) / 32);
  build_planes_kernel<<<(unsigned)blocks, 256, 0, st>>>(lat, pow, lpT, d, flag);
  plane_min_kernel<<<(d.M * 2 * d.B + 3) / 4, 128, 0, st>>>(lpT, d, pmin);
  return 2;
}
