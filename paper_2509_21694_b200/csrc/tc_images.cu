#include "tc_images.cuh"

namespace {
__global__ void k_edge_images(const float* __restrict__ W2, const float* __restrict__ W1c, int d,
                              __half* __restrict__ W2img, __half* __restrict__ W1cimg) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < d * d) {
    const int o = idx / d, i = idx % d;
    W2img[tc_sw128_index(d, o, i)] = __float2half_rn(0.5f * W2[idx]);
  }
  if (idx < d * 16) {
    const int c = idx / 16, k = idx % 16;
    W1cimg[tc_nosw_index(16, c, k)] = __float2half_rn(0.5f * W1c[idx]);
  }
}
__device__ void split3_store(float x, __nv_bfloat16* dst, size_t stride) {
  for (int t = 0; t < 3; ++t) {
    const __nv_bfloat16 h = __float2bfloat16_rn(x);
    dst[t * stride] = h;
    x -= __bfloat162float(h);
  }
}
__global__ void k_edge_images_x3(const float* __restrict__ W2, const float* __restrict__ W1c, const float* __restrict__ W3, int d,
                                 __nv_bfloat16* __restrict__ W2x3, __nv_bfloat16* __restrict__ W13x3) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < d * d) split3_store(W2[idx], W2x3 + tc_sw128_index(d, idx / d, idx % d), (size_t)d * d);
  if (idx < d * 32) {
    const int c = idx / 32, k = idx % 32;
    const float x = k < 16 ? W1c[c * 16 + k] : (W3 ? W3[c * 16 + k - 16] : 0.f);
    split3_store(x, W13x3 + tc_nosw_index(32, c, k), (size_t)d * 32);
  }
}
}  // namespace

void mlip_make_edge_images(cudaStream_t st, const float* W2, const float* W1c, int d, __half* W2img, __half* W1cimg) {
  k_edge_images<<<(d * d + 255) / 256, 256, 0, st>>>(W2, W1c, d, W2img, W1cimg);
}
void mlip_make_edge_images_x3(cudaStream_t st, const float* W2, const float* W1c, const float* W3, int d, __nv_bfloat16* W2x3,
                              __nv_bfloat16* W13x3) {
  k_edge_images_x3<<<(d * d + 255) / 256, 256, 0, st>>>(W2, W1c, W3, d, W2x3, W13x3);
}
