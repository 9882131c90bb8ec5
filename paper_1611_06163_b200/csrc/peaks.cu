// peaks.cu — measured denominators of the pair kernel's roofline ("measure with an FFMA microbenchmark",
// "BW_L2 ... microbenchmark (read-only sweep of a 32 MB buffer)"): tdpd_measure_peaks.  Not on the timed path.
//   FP32:  independent FMA chains, 16 resident warps per SM, once with scalar fma.rn.f32 (three register operands:
//          the register file delivers ~2.1 of the 4 warp instructions per clock and SM) and once with the packed
//          fma.rn.f32x2 of sm_100 (FFMA2 in SASS: ~1.8 warp instructions per clock and SM, two FMAs per lane each);
//          the larger of the two is the FP32 peak the roofline uses.
//   L2:    read-only sweep of a 32 MB buffer (ld.global.cg, 16 B per lane), repeated; the buffer stays L2-resident.
//   HBM:   the same sweep over 1 GiB.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tdpd.h"

namespace {

template <bool PACKED>
__global__ void __launch_bounds__(256, 2) k_peak_fma(float* out, uint32_t seed, int iters) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  float a0 = 1.f + t * 1e-9f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f,
        a7 = a0 + 7.f;
  const float b = 1.0000001f + seed * 1e-9f, c = 1e-9f + seed * 1e-12f, b2 = 0.99999f - seed * 1e-9f,
              c2 = 2e-9f + seed * 1e-12f;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      if (PACKED) {  // 8 packed instructions = 16 FMAs per lane
        asm volatile(
            "{.reg .b64 x0,x1,x2,x3,y,z;\n\t"
            "mov.b64 x0,{%0,%1};mov.b64 x1,{%2,%3};mov.b64 x2,{%4,%5};mov.b64 x3,{%6,%7};mov.b64 y,{%8,%9};mov.b64 z,{%10,%11};\n\t"
            "fma.rn.f32x2 x0,x0,y,z;fma.rn.f32x2 x1,x1,y,z;fma.rn.f32x2 x2,x2,y,z;fma.rn.f32x2 x3,x3,y,z;\n\t"
            "fma.rn.f32x2 x0,x0,y,z;fma.rn.f32x2 x1,x1,y,z;fma.rn.f32x2 x2,x2,y,z;fma.rn.f32x2 x3,x3,y,z;\n\t"
            "mov.b64 {%0,%1},x0;mov.b64 {%2,%3},x1;mov.b64 {%4,%5},x2;mov.b64 {%6,%7},x3;}"
            : "+f"(a0), "+f"(a1), "+f"(a2), "+f"(a3), "+f"(a4), "+f"(a5), "+f"(a6), "+f"(a7)
            : "f"(b), "f"(b2), "f"(c), "f"(c2));
      } else {  // 8 scalar FMAs per lane
        a0 = fmaf(a0, b, c); a1 = fmaf(a1, b2, c2); a2 = fmaf(a2, b, c2); a3 = fmaf(a3, b2, c);
        a4 = fmaf(a4, b, c); a5 = fmaf(a5, b2, c2); a6 = fmaf(a6, b, c2); a7 = fmaf(a7, b2, c);
      }
    }
  }
  out[t] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}

__global__ void __launch_bounds__(256) k_peak_read(const float4* __restrict__ buf, size_t n4, int reps, float* out) {
  float4 acc = make_float4(0, 0, 0, 0);
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (int r = 0; r < reps; ++r)
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
      float4 v;
      asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(buf + i));
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
  if (acc.x + acc.y + acc.z + acc.w == 123.456f) out[0] = acc.x;  // keeps the loads
}

template <bool PACKED>
bool time_fma(int nsm, float* out, double* tflops) {
  const int nblk = 2 * nsm, iters = 40000;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  k_peak_fma<PACKED><<<nblk, 256>>>(out, 1, iters / 8);
  cudaEventRecord(e0);
  k_peak_fma<PACKED><<<nblk, 256>>>(out, 2, iters);
  cudaEventRecord(e1);
  bool ok = cudaDeviceSynchronize() == cudaSuccess;
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (!ok || ms <= 0.f) return false;
  const double fma_per_lane = (double)iters * 4 * (PACKED ? 16 : 8);
  *tflops = fma_per_lane * 2.0 * 256.0 * nblk / (ms * 1e-3) / 1e12;
  return true;
}

bool time_read(size_t bytes, int reps, int nsm, float* out, double* gbs) {
  float4* buf = nullptr;
  if (cudaMalloc(&buf, bytes) != cudaSuccess) return false;
  cudaMemset(buf, 0, bytes);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  k_peak_read<<<nsm * 8, 256>>>(buf, bytes / 16, 2, out);
  cudaEventRecord(e0);
  k_peak_read<<<nsm * 8, 256>>>(buf, bytes / 16, reps, out);
  cudaEventRecord(e1);
  bool ok = cudaDeviceSynchronize() == cudaSuccess;
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(buf);
  if (!ok || ms <= 0.f) return false;
  *gbs = (double)bytes * reps / (ms * 1e-3) / 1e9;
  return true;
}
}  // namespace

extern "C" int tdpd_measure_peaks(int device, tdpd_peaks* out) {
  if (!out) return TDPD_EINVAL;
  if (cudaSetDevice(device) != cudaSuccess) return TDPD_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return TDPD_ECUDA;
  const int nsm = prop.multiProcessorCount;
  float* o = nullptr;
  if (cudaMalloc(&o, (size_t)nsm * 8 * 256 * 4) != cudaSuccess) return TDPD_ENOMEM;
  bool ok = time_fma<false>(nsm, o, &out->fp32_fma_tflops) && time_fma<true>(nsm, o, &out->fp32_fma2_tflops) &&
            time_read((size_t)32 << 20, 2000, nsm, o, &out->l2_read_gbs) &&
            time_read((size_t)1 << 30, 50, nsm, o, &out->hbm_read_gbs);
  out->n_sm = nsm;
  cudaFree(o);
  return ok ? TDPD_OK : TDPD_ECUDA;
}
