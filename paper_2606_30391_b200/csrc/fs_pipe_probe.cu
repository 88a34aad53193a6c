// fs_pipe_probe.cu — measurement only: per-SM issue rates of the instruction classes the path is made of
// (DESIGN.md section 7 derives the "alu" roofline peak from them).  Each kernel runs a long, fully unrolled chain
// of ONE instruction class on 8 independent accumulators per thread, 1024 threads per SM on every SM, and is
// timed with CUDA events; rate = thread-instructions / (time x SM clock x SMs).
#include "fs_kernels.h"

namespace {

constexpr int PP_ITERS = 4096, PP_ILP = 8;

template <int OP>
__global__ void __launch_bounds__(1024) pipe_kernel(float* out, float seed) {
  float a[PP_ILP]; int b[PP_ILP];
#pragma unroll
  for (int i = 0; i < PP_ILP; ++i) { a[i] = seed + threadIdx.x * 1e-3f + i; b[i] = (int)threadIdx.x + i; }
  const float c = seed * 1.0001f, dd = seed + 0.5f;
  for (int it = 0; it < PP_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PP_ILP; ++i) {
      if (OP == 0) a[i] = __fmul_rn(a[i], c);                                   // FMUL
      if (OP == 1) a[i] = __fadd_rn(a[i], c);                                   // FADD
      if (OP == 2) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(dd));  // FMNMX
      if (OP == 3) asm volatile("{.reg .pred p; setp.le.f32 p, %0, %1; @p min.f32 %0, %0, %2;}"
                                : "+f"(a[i]) : "f"(c), "f"(dd));                // FSETP + predicated FMNMX
      if (OP == 4) asm volatile("min.s32 %0, %0, %1;" : "+r"(b[i]) : "r"(it));  // IMNMX
      if (OP == 5) asm volatile("{.reg .pred p; setp.le.s32 p, %0, %1; selp.s32 %0, %0, %2, p;}"
                                : "+r"(b[i]) : "r"(it), "r"(i));                // ISETP + SEL
      if (OP == 6) asm volatile("{.reg .u32 m; set.gt.u32.f32 m, %1, %2; or.b32 m, m, %3; min.u32 %0, %0, m;}"
                                : "+r"(b[i]) : "f"(a[i]), "f"(c), "r"(it));     // FSET mask + LOP3 + unsigned min
    }
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PP_ILP; ++i) s += a[i] + (float)b[i];
  if (s == 123.456f) out[0] = s;      // keeps the chains alive
}

template <int OP>
double run_pipe(float* d_out, int sms, double sm_hz, int per_iter) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  pipe_kernel<OP><<<sms, 1024>>>(d_out, 1.0f);
  cudaEventRecord(e0);
  pipe_kernel<OP><<<sms, 1024>>>(d_out, 1.0f);
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  const double insts = (double)sms * 1024.0 * PP_ITERS * PP_ILP * per_iter;
  return insts / (ms * 1e-3 * sm_hz * sms);        // thread-instructions per clock per SM
}

}  // namespace

// out[7]: FMUL, FADD, FMNMX, FSETP+@FMNMX (per instruction), IMNMX, ISETP+SEL (per instruction),
//         FSET mask + OR + unsigned min (per instruction)
extern "C" int fs_probe_pipe_rates(int cuda_device, double sm_mhz, double* out) {
  if (!out || sm_mhz <= 0) return FS_ERR_ARG;
  if (cudaSetDevice(cuda_device) != cudaSuccess) { cudaGetLastError(); return FS_ERR_CUDA; }
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device);
  float* d_out = nullptr;
  if (cudaMalloc(&d_out, 16) != cudaSuccess) { cudaGetLastError(); return FS_ERR_NOMEM; }
  const double hz = sm_mhz * 1e6;
  out[0] = run_pipe<0>(d_out, sms, hz, 1); out[1] = run_pipe<1>(d_out, sms, hz, 1);
  out[2] = run_pipe<2>(d_out, sms, hz, 1); out[3] = run_pipe<3>(d_out, sms, hz, 2);
  out[4] = run_pipe<4>(d_out, sms, hz, 1); out[5] = run_pipe<5>(d_out, sms, hz, 2);
  out[6] = run_pipe<6>(d_out, sms, hz, 3);
  cudaFree(d_out);
  return cudaGetLastError() == cudaSuccess ? FS_OK : FS_ERR_CUDA;
}
