// fs_alg1.cu — Algorithm 1, phase 1 and the Energy Waste Ratio (Eq. 5-7).
//
// fs_llm_profile: per active LLM, from its average input / output length,
//   (SM_p, F_p), (SM_d, F_d) = LUT argmin of the prefill / decode energy under the TTFT / TBT SLO
//   (ties: lowest phi, then lowest sigma: key flat = phi*S + sigma);
//   SM_l = (SM_p*T_p + SM_d*T_d)/(T_p + T_d) (Eq. 8);  l.S = ceil(SM_l);  l.F = argmin over phi of the
//   total energy at l.S units with both SLOs met;  M_l = Weights + lambda*W*Size_KV (Little's law).
//   One warp per LLM: lanes over the (sigma, phi) plane (coalesced in the plane layout), 64-bit
//   (energy, flat) keys reduced by shuffles; then lanes over phi for l.F.
// fs_ewr: F_g = max F_l per GPU (atomicMax on the bit patterns of positive floats), then
//   E_waste = sum t_l (F_g^3 - F_l^3), E_optimal = sum t_l F_l^3 in binary64 (one block, fixed tree).
#include "fs_kernels.h"

namespace {

__global__ void __launch_bounds__(128) llm_profile_kernel(FsView v, int n, const fs_llm* __restrict__ llms,
                                                         fs_llm_profile* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int li = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (li >= n) return;
  const FsDimsDev d = v.d;
  const fs_llm l = llms[li];
  fs_llm_profile o;
  o.sigma_p = o.phi_p = o.sigma_d = o.phi_d = o.need_units = o.phi_l = -1;
  o.t_p_ms = o.t_d_ms = o.p_p_w = o.p_d_w = o.sm_units = o.t_l_ms = o.e_l_mj = o.mem_mb = FS_INF; o._pad = 0;
  if (l.model < 0 || l.model >= d.M || l.avg_in >= (1u << 24) || l.avg_out >= (1u << 24)) {
    if (lane == 0) { fs_raise(v.flag, FS_FLAG_REQUEST); out[li] = o; }
    return;
  }
  const int m = l.model;
  const uint32_t L = l.avg_in, O = l.avg_out;
  const uint32_t n0 = L < (uint32_t)d.B ? L : (uint32_t)d.B;
  const int br0 = n0 ? (int)n0 - 1 : 0;
  const uint32_t rounds0 = n0 ? fs_ceil_div(L, n0) : 0u;
  const float2* lp0 = v.lpT + fs_plane(d, m, 0, br0);    // {LAT, POW} planes of the prefill bucket and of decode bucket 0
  const float2* lp1 = v.lpT + fs_plane(d, m, 1, 0);
  // ---- preferred configuration per phase --------------------------------------------------------
  unsigned long long kp = FS_KEY_NONE, kd = FS_KEY_NONE;
  for (int x = lane; x < d.S * d.F; x += 32) {          // x = sigma*F + phi (plane order)
    const int sg = x / d.F, phi = x % d.F;
    const uint32_t flat = (uint32_t)(phi * d.S + sg);
    FsSlot a; a.ok = true; a.t = 0.f; a.e = 0.f;
    if (L > 0) a = fs_slot(0, lp0[x].x, lp0[x].y, rounds0, 0.0f, l.slo_ttft_ms);
    if (a.ok && a.e < FS_INF) { const unsigned long long k = fs_make_key(a.e, flat); kp = k < kp ? k : kp; }
    FsSlot b; b.ok = true; b.t = 0.f; b.e = 0.f;
    if (O > 0) b = fs_slot(1, lp1[x].x, lp1[x].y, O, 0.0f, l.slo_tbt_ms);
    if (b.ok && b.e < FS_INF) { const unsigned long long k = fs_make_key(b.e, flat); kd = k < kd ? k : kd; }
  }
  kp = fs_warp_min_key(kp); kd = fs_warp_min_key(kd);
  if (kp != FS_KEY_NONE) {
    const int flat = (int)(uint32_t)kp, phi = flat / d.S, sg = flat % d.S, x = sg * d.F + phi;
    o.sigma_p = (int16_t)sg; o.phi_p = (int16_t)phi;
    o.t_p_ms = L ? __fmul_rn(__uint2float_rn(rounds0), lp0[x].x) : 0.0f; o.p_p_w = L ? lp0[x].y : 0.0f;
  }
  if (kd != FS_KEY_NONE) {
    const int flat = (int)(uint32_t)kd, phi = flat / d.S, sg = flat % d.S, x = sg * d.F + phi;
    o.sigma_d = (int16_t)sg; o.phi_d = (int16_t)phi;
    o.t_d_ms = O ? __fmul_rn(__uint2float_rn(O), lp1[x].x) : 0.0f; o.p_d_w = O ? lp1[x].y : 0.0f;
  }
  if (kp != FS_KEY_NONE && kd != FS_KEY_NONE) {
    // ---- Eq. 8, l.S, l.F, Little's law -----------------------------------------------------------
    const float tsum = __fadd_rn(o.t_p_ms, o.t_d_ms);
    o.sm_units = tsum > 0.0f
        ? __fdiv_rn(__fadd_rn(__fmul_rn((float)(o.sigma_p + 1), o.t_p_ms), __fmul_rn((float)(o.sigma_d + 1), o.t_d_ms)), tsum)
        : 1.0f;
    int need = (int)ceilf(o.sm_units);
    need = need < 1 ? 1 : (need > d.S ? d.S : need);
    o.need_units = (int16_t)need;
    unsigned long long kl = FS_KEY_NONE;
    for (int phi = lane; phi < d.F; phi += 32) {
      const int x = (need - 1) * d.F + phi;
      FsSlot a; a.ok = true; a.t = 0.f; a.e = 0.f;
      if (L > 0) a = fs_slot(0, lp0[x].x, lp0[x].y, rounds0, 0.0f, l.slo_ttft_ms);
      FsSlot b; b.ok = true; b.t = 0.f; b.e = 0.f;
      if (O > 0) b = fs_slot(1, lp1[x].x, lp1[x].y, O, 0.0f, l.slo_tbt_ms);
      const float e = __fadd_rn(a.e, b.e);
      if (a.ok && b.ok && e < FS_INF) { const unsigned long long k = fs_make_key(e, (uint32_t)phi); kl = k < kl ? k : kl; }
    }
    kl = fs_warp_min_key(kl);
    if (kl != FS_KEY_NONE) {
      const int phi = (int)(uint32_t)kl, x = (need - 1) * d.F + phi;
      const float tp = L ? __fmul_rn(__uint2float_rn(rounds0), lp0[x].x) : 0.0f;
      const float td = O ? __fmul_rn(__uint2float_rn(O), lp1[x].x) : 0.0f;
      o.phi_l = (int16_t)phi; o.t_l_ms = __fadd_rn(tp, td); o.e_l_mj = fs_unorderable((uint32_t)(kl >> 32));
      const float nconc = __fmul_rn(l.lambda_rps, __fdiv_rn(o.t_l_ms, 1000.0f));
      const float kvsize = __fmul_rn(__uint2float_rn(L + O), v.models[m].kv_mb_per_token);
      o.mem_mb = __fadd_rn(v.models[m].weights_mb, __fmul_rn(nconc, kvsize));
    }
  }
  if (lane == 0) out[li] = o;
}

__global__ void ewr_fmax_kernel(int n, const int32_t* __restrict__ gpu_of, const float* __restrict__ f_mhz, int K,
                                float* __restrict__ fg, int* flag) {
  const int l = blockIdx.x * blockDim.x + threadIdx.x;
  if (l >= n) return;
  const int g = gpu_of[l];
  if (g < 0) return;
  if (g >= K) { fs_raise(flag, FS_FLAG_ARG); return; }
  const float f = f_mhz[l];
  if (f > 0.0f) atomicMax(reinterpret_cast<int*>(fg) + g, __float_as_int(f));   // positive floats order like ints
}

__global__ void __launch_bounds__(1024) ewr_sum_kernel(int n, const int32_t* __restrict__ gpu_of,
                                                      const float* __restrict__ f_mhz, const float* __restrict__ t_ms,
                                                      int K, const float* __restrict__ fg, double* __restrict__ out3) {
  __shared__ double sw[1024], so[1024];
  double w = 0.0, o = 0.0;
  for (int l = threadIdx.x; l < n; l += 1024) {
    const int g = gpu_of[l];
    if (g < 0 || g >= K) continue;
    const double F = fg[g], f = f_mhz[l], t = t_ms[l];
    w += t * (F * F * F - f * f * f);
    o += t * (f * f * f);
  }
  sw[threadIdx.x] = w; so[threadIdx.x] = o;
  __syncthreads();
  for (int s = 512; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) { sw[threadIdx.x] += sw[threadIdx.x + s]; so[threadIdx.x] += so[threadIdx.x + s]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out3[0] = sw[0]; out3[1] = so[0]; out3[2] = so[0] > 0.0 ? sw[0] / so[0] : 0.0; }
}

}  // namespace

int fsk_llm_profile(const FsView& v, int n, const fs_llm* llms, fs_llm_profile* out, cudaStream_t st) {
  if (n <= 0) return 0;
  llm_profile_kernel<<<(n + 3) / 4, 128, 0, st>>>(v, n, llms, out);
  return 1;
}

int fsk_ewr(int n, const int32_t* gpu_of, const float* f_mhz, const float* t_ms, int K, float* fg, double* out3,
            int* flag, cudaStream_t st) {
  if (K > 0) cudaMemsetAsync(fg, 0, sizeof(float) * (size_t)K, st);
  if (n > 0) ewr_fmax_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, gpu_of, f_mhz, K, fg, flag);
  ewr_sum_kernel<<<1, 1024, 0, st>>>(n, gpu_of, f_mhz, t_ms, K, fg, out3);
  return n > 0 ? 2 : 1;
}
