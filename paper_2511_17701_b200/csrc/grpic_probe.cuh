// grpic_probe.cuh — register-only throughput probes: the denominators of the ALU roofline.
//
// One launch = grid x 256 threads, each running kChains independent dependent-chains of one instruction kind for
// `iters` rounds: FFMA (FP32 peak = 2 flop per lane and cycle), DFMA (FP64), MUFU.RSQ (special-function unit) and
// red.shared-free plain LDS+FADD+STS read-modify-writes of a lane-private shared word (what the lane windows of
// k_step_lanes do).  bench.py times the launch with CUDA events and divides the returned operation count by it.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace grpic {

constexpr int kProbeChains = 8;
constexpr int kProbeBlock = 256;

template <int kKind>
__global__ void __launch_bounds__(kProbeBlock) k_probe(int iters, float seed, float* out) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (kKind == 0) {                      // FFMA
    float x[kProbeChains];
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) x[c] = seed + (float)(t + c) * 1e-9f;
    const float a = 1.0f - 1e-7f * seed, b = 1e-9f * seed;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) x[c] = fmaf(x[c], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) s += x[c];
    if (s == 12345.678f) out[0] = s;
  } else if (kKind == 1) {               // DFMA
    double x[kProbeChains];
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) x[c] = (double)seed + (double)(t + c) * 1e-12;
    const double a = 1.0 - 1e-9 * seed, b = 1e-12 * seed;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) x[c] = fma(x[c], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) s += x[c];
    if (s == 12345.678) out[0] = (float)s;
  } else if (kKind == 2) {               // MUFU.RSQ
    float x[kProbeChains];
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) x[c] = 1.0f + seed + (float)(t + c) * 1e-6f;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x[c]));
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) s += x[c];
    if (s == 12345.678f) out[0] = s;
  } else {                               // lane-private shared read-modify-write (LDS + FADD + STS), 8 slots per lane
    __shared__ float w[kProbeChains * kProbeBlock];
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) w[c * kProbeBlock + threadIdx.x] = seed;
    volatile float* v = w;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) v[c * kProbeBlock + threadIdx.x] = v[c * kProbeBlock + threadIdx.x] + seed;
    }
    if (w[threadIdx.x] == 12345.678f) out[0] = w[threadIdx.x];
  }
}

}  // namespace grpic
