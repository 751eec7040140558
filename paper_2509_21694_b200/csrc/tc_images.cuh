// f16 shared-memory operand images used by the tcgen05 edge kernels. The images are stored in
// global memory in exactly the byte order the kernels want in shared memory, so a CTA stages them
// with one linear bulk copy (cp.async.bulk) and no tensor map.
//
// Canonical UMMA layouts (units: 16-bit elements; a "chunk" is 8 elements = 16 bytes):
//  * K-major, 128-byte swizzle, operand [R rows x K]: K is cut into blocks of 64 (128 bytes);
//    block kb is a dense [R x 64] slab at element offset kb*R*64; inside it element (r, k) sits
//    at r*64 + ((k/8) ^ (r%8))*8 + k%8. Descriptor: SBO = 1024 B (8 rows), layout SWIZZLE_128B;
//    one MMA (K=16) advances the start address by 32 B inside the slab. The SAME bytes read as
//    an MN-major operand [MN = 64-wide blocks, K = rows] use LBO = slab stride, SBO = 1024 B.
//  * K-major, no swizzle, operand [R rows x K]: 8x8 core matrices of 128 contiguous bytes;
//    element (r, k) at (r/8)*SBO_e + (k/8)*LBO_e + (r%8)*8 + k%8 with LBO_e = 64 (128 B) and
//    SBO_e = (K/8)*64.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

__host__ __device__ inline int tc_sw128_index(int rows, int r, int k) {
  return (k >> 6) * rows * 64 + r * 64 + ((((k & 63) >> 3) ^ (r & 7)) << 3) + (k & 7);
}
__host__ __device__ inline int tc_nosw_index(int K, int r, int k) {
  return (r >> 3) * (K >> 3) * 64 + (k >> 3) * 64 + (r & 7) * 8 + (k & 7);
}

// The edge kernels evaluate SiLU(2x) = x + x tanh(x) on HALVED pre-activations, so the operands
// that produce pre-activations carry an exact factor 1/2:
// W2 [d,d] row-major [out,in] -> W2img  : SW128 K-major, rows = out, K = in, values W2/2
//                                         (read MN-major for the adjoint pbar . W2)
// W1c [d,16] (padded)         -> W1cimg : no-swizzle K-major, rows = channel, K = 16, values W1c/2
//                                         (read MN-major, N = rbf index, K = channel, for ebar = abar . W1c)
void mlip_make_edge_images(cudaStream_t st, const float* W2, const float* W1c, int d, __half* W2img, __half* W1cimg);

// fp32 path on the tensor cores (edge_x3.cu): x = x1 + x2 + x3, x1 = bf16(x), x2 = bf16(x - x1), x3 = bf16(x - x1 - x2).
// W2x3  [3][d*d]  : the three terms of W2 (not halved), each in the SW128 K-major layout of W2img
// W13x3 [3][d*32] : the three terms of [W1c | W3] [d,32] (W3 = 0 when null), no-swizzle K-major, rows = channel, K = 32
void mlip_make_edge_images_x3(cudaStream_t st, const float* W2, const float* W1c, const float* W3, int d, __nv_bfloat16* W2x3,
                              __nv_bfloat16* W13x3);
