// Scalar device math shared by the kernels: SiLU and its derivative (O3/O5), cosine envelope and
// Gaussian radial basis with derivatives (O2).
#pragma once
#include <cuda_runtime.h>

__device__ __forceinline__ float sigmoid_f(float x) { return __fdividef(1.0f, 1.0f + __expf(-x)); }
__device__ __forceinline__ float silu_f(float x) { return x * sigmoid_f(x); }
// SiLU'(x) = s (1 + x (1 - s))
__device__ __forceinline__ float dsilu_f(float x) {
  const float s = sigmoid_f(x);
  return s * fmaf(x, 1.0f - s, 1.0f);
}
__device__ __forceinline__ void silu_both_f(float x, float& y, float& dy) {
  const float s = sigmoid_f(x);
  y = x * s;
  dy = s * fmaf(x, 1.0f - s, 1.0f);
}

// u(r) = (cos(pi r / rc) + 1)/2, u'(r) = -(pi / 2 rc) sin(pi r / rc)
__device__ __forceinline__ void envelope_f(float r, float r_cut, float& u, float& du) {
  float s, c;
  sincospif(r / r_cut, &s, &c);
  u = 0.5f * (c + 1.0f);
  du = -(1.5707963267948966f / r_cut) * s;
}
// g_k(r) = exp(-gamma (r - k Delta)^2), Delta = rc/(n_rbf-1), gamma = 1/(2 Delta^2)
__device__ __forceinline__ void rbf_f(float r, float r_cut, int n_rbf, int k, float& g, float& dg) {
  const float delta = r_cut / (float)(n_rbf - 1);
  const float gamma = 0.5f / (delta * delta);
  const float diff = r - (float)k * delta;
  g = expf(-gamma * diff * diff);
  dg = -2.0f * gamma * diff * g;
}

// SiLU through the hardware tanh (MUFU.TANH, abs. error ~2^-11): used by the MLIP_BF16 kernels only,
// where every result is rounded to bf16 (ulp 2^-8) anyway. sigma(x) = 1/2 + 1/2 tanh(x/2).
__device__ __forceinline__ float tanh_approx_f(float x) {
  float y;
  asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float silu_tanh_f(float x) {
  const float h = 0.5f * x;
  return fmaf(h, tanh_approx_f(h), h);
}
__device__ __forceinline__ void silu_both_tanh_f(float x, float& y, float& dy) {
  const float s = fmaf(0.5f, tanh_approx_f(0.5f * x), 0.5f);
  y = x * s;
  dy = fmaf(y, 1.0f - s, s);  // s (1 + x (1 - s))
}
