// fp32 CUDA-core node-level GEMM with fused prologue / epilogue (steps A8, A9 and their adjoints
// in the MLIP_FP32 path): Y[n,N] = epi( act(X)[n,K] . B^T + bias ), X = [X1 | X2].
// 64x64 output tile, K step 16, 256 threads, 4x4 register block per thread.
#include <stdlib.h>
#include <string.h>
#include "common.cuh"
#include "mathfn.cuh"

namespace {
constexpr int BM = 64, BN = 64, BK = 16;

__global__ void __launch_bounds__(256) k_gemm_f32(GemmArgs a) {
  __shared__ __align__(16) float As[BK][BM + 4];
  __shared__ __align__(16) float Bs[BK][BN + 4];
  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;
  const int64_t row0 = (int64_t)blockIdx.x * BM;
  const int col0 = blockIdx.y * BN;
  const int K = a.K1 + a.K2;
  const float* Bw = (const float*)a.B;
  const int lr = tid >> 2, lk = (tid & 3) * 4;  // loader: row lr, k offset lk..lk+3
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < K; k0 += BK) {
    float4 av = make_float4(0.f, 0.f, 0.f, 0.f);
    const int64_t r = row0 + lr;
    if (r < a.n) {
      const int kk = k0 + lk;
      const float* src = kk < a.K1 ? a.X1 + r * a.ld1 + kk : a.X2 + r * a.ld2 + (kk - a.K1);
      av = *reinterpret_cast<const float4*>(src);
      if (a.act_in) { av.x = silu_f(av.x); av.y = silu_f(av.y); av.z = silu_f(av.z); av.w = silu_f(av.w); }
    }
    const float4 bv = *reinterpret_cast<const float4*>(Bw + (size_t)(col0 + lr) * K + k0 + lk);
    __syncthreads();
    As[lk + 0][lr] = av.x; As[lk + 1][lr] = av.y; As[lk + 2][lr] = av.z; As[lk + 3][lr] = av.w;
    Bs[lk + 0][lr] = bv.x; Bs[lk + 1][lr] = bv.y; Bs[lk + 2][lr] = bv.z; Bs[lk + 3][lr] = bv.w;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      const float4 x = *reinterpret_cast<const float4*>(&As[k][ty * 4]);
      const float4 w = *reinterpret_cast<const float4*>(&Bs[k][tx * 4]);
      const float xs[4] = {x.x, x.y, x.z, x.w}, ws[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(xs[i], ws[j], acc[i][j]);
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t r = row0 + ty * 4 + i;
    if (r >= a.n) continue;
    const int c = col0 + tx * 4;
    float y[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) y[j] = acc[i][j] + (a.bias ? a.bias[c + j] : 0.f);
    if (a.mul_dsilu) {
      const float4 z = *reinterpret_cast<const float4*>(a.mul_dsilu + r * a.ldz + c);
      y[0] *= dsilu_f(z.x); y[1] *= dsilu_f(z.y); y[2] *= dsilu_f(z.z); y[3] *= dsilu_f(z.w);
    }
    if (a.residual) {
      const float4 q = *reinterpret_cast<const float4*>(a.residual + r * a.ldr + c);
      y[0] += q.x; y[1] += q.y; y[2] += q.z; y[3] += q.w;
    }
    if (a.Y) *reinterpret_cast<float4*>(a.Y + r * a.ldy + c) = make_float4(y[0], y[1], y[2], y[3]);
    if (a.Ybf) {
      __nv_bfloat162 p0 = __floats2bfloat162_rn(y[0], y[1]), p1 = __floats2bfloat162_rn(y[2], y[3]);
      uint2 pk;
      pk.x = *reinterpret_cast<uint32_t*>(&p0); pk.y = *reinterpret_cast<uint32_t*>(&p1);
      *reinterpret_cast<uint2*>(a.Ybf + r * a.ldy + c) = pk;
    }
  }
}
}  // namespace

int mlip_gemm_f32(mlip_ctx* ctx, const GemmArgs& a) {
  if (a.n <= 0) return MLIP_OK;
  // d = 128: on the tensor cores (node_x3.cu) unless MLIP_B200_FP32_EDGE=cuda asks for the CUDA-core kernels (A/B runs)
  static const bool cuda_cores = [] { const char* v = getenv("MLIP_B200_FP32_EDGE"); return v && !strcmp(v, "cuda"); }();
  if (!cuda_cores && !ctx->x3_img.empty() && mlip_gemm_x3_supported(a)) {
    auto it = ctx->x3_img.find(a.B);
    if (it != ctx->x3_img.end()) return mlip_gemm_x3(ctx, a, it->second);
  }
  if (a.N % BN || a.K1 % BK || a.K2 % BK) { ctx->set_error("gemm_f32: shape not a multiple of the tile"); return MLIP_ERR_UNSUPPORTED; }
  dim3 grid((unsigned)((a.n + BM - 1) / BM), a.N / BN);
  k_gemm_f32<<<grid, 256, 0, ctx->stream>>>(a);
  ctx->launches++;
  return MLIP_OK;
}
