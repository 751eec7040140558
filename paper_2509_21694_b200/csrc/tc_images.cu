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
}  // namespace

void mlip_make_edge_images(cudaStream_t st, const float* W2, const float* W1c, int d, __half* W2img, __half* W1cimg) {
  k_edge_images<<<(d * d + 255) / 256, 256, 0, st>>>(W2, W1c, d, W2img, W1cimg);
}
