// fs_tables.cu — fs_load_profiles device work: validate the LUT and build the
// plane layout [M][2][B][S][F] in which the (sigma,phi) plane of one (model, phase, batch
// bucket) is one contiguous S*F*4-byte block (what placement stages per request).
#include "fs_kernels.h"

namespace {

// One block transposes a 32x32 (phi, beta) tile of one (model, phase, sigma) slice for both
// tables.  Reads are coalesced along beta, writes along phi.
__global__ void __launch_bounds__(256) build_planes_kernel(const float* __restrict__ lat,
                                                          const float* __restrict__ pow,
                                                          float* __restrict__ latT,
                                                          float* __restrict__ powT, FsDimsDev d,
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
      latT[o] = tl[tx][r];
      powT[o] = tp[tx][r];
    }
  }
  if (bad) fs_raise(flag, FS_FLAG_TABLE);
}

// dmin[m][b][s] = { min LAT, min POW } of the decode plane (m, 1, b) over shares <= s and all phi: the
// bounds l1_min / p1_min of a warm (GPU, slot) item are then one lookup at (model, bucket, sm_free - 1)
__global__ void __launch_bounds__(128) decode_min_kernel(const float* __restrict__ latT, const float* __restrict__ powT,
                                                        FsDimsDev d, float2* __restrict__ dmin) {
  const int lane = threadIdx.x & 31;
  const int w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (w >= d.M * d.B) return;
  const int m = w / d.B, b = w % d.B;
  const float* pl = latT + fs_plane(d, m, 1, b); const float* pp = powT + fs_plane(d, m, 1, b);
  float ml = FS_INF, mp = FS_INF;
  for (int s = 0; s < d.S; ++s) {
    float l = FS_INF, p = FS_INF;
    for (int phi = lane; phi < d.F; phi += 32) { l = fminf(l, pl[s * d.F + phi]); p = fminf(p, pp[s * d.F + phi]); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      l = fminf(l, __shfl_xor_sync(0xffffffffu, l, o)); p = fminf(p, __shfl_xor_sync(0xffffffffu, p, o));
    }
    ml = fminf(ml, l); mp = fminf(mp, p);
    if (lane == 0) dmin[(size_t)w * d.S + s] = make_float2(ml, mp);
  }
}

}  // namespace

int fsk_build_planes(const float* lat, const float* pow, float* latT, float* powT, float2* dmin, FsDimsDev d,
                     int* flag, cudaStream_t st) {
  const long long blocks = (long long)d.M * 2 * d.S * ((d.F + 31) / 32) * ((d.B + 31) / 32);
  build_planes_kernel<<<(unsigned)blocks, 256, 0, st>>>(lat, pow, latT, powT, d, flag);
  decode_min_kernel<<<(d.M * d.B + 3) / 4, 128, 0, st>>>(latT, powT, d, dmin);
  return 2;
}
