// bf16 tensor-core node-level GEMM with fused prologue / epilogue (steps A8, A9 and their adjoints
// in the MLIP_BF16 path): Y[n,N] = epi( act(X)[n,K] . B^T + bias ), X = [X1 | X2] fp32 in global.
//
// One CTA owns 128 rows and the full output width N (= d). K is streamed in chunks of 64: the
// threads convert the fp32 activations to bf16 (optionally through SiLU) straight into a K-major
// SWIZZLE_128B operand slab, the matching [N x 64] slab of the bf16 weight is staged with
// cp.async, and one thread issues four tcgen05.mma (M=128, N, K=16) into a TMEM accumulator.
// Two stages: the conversion of chunk k+1 overlaps the MMAs of chunk k (tcgen05.commit -> mbarrier
// frees a stage). Epilogue: tcgen05.ld -> bias / SiLU' / residual -> fp32 or bf16 rows.
#include "common.cuh"
#include "mathfn.cuh"
#include "tc_ptx.cuh"

namespace {
constexpr int BM = 128, BK = 64;

template <int N>
struct NodeSmem {
  static constexpr uint32_t a_bytes = BM * BK * 2;  // 16 KB
  static constexpr uint32_t b_bytes = N * BK * 2;   // 32 KB at N = 256
  static constexpr uint32_t a_off(int s) { return s * a_bytes; }
  static constexpr uint32_t b_off(int s) { return 2 * a_bytes + s * b_bytes; }
  static constexpr uint32_t bar_off = 2 * a_bytes + 2 * b_bytes;
  static constexpr uint32_t bytes = bar_off + 64 + 1024;  // + alignment slack
};

template <int N>
__global__ void __launch_bounds__(256) k_gemm_bf16(GemmArgs a) {
  extern __shared__ unsigned char smem_raw[];
  using SM = NodeSmem<N>;
  // SWIZZLE_128B operands need 1024-byte aligned slabs
  const uint32_t base = (tc::smem_u32(smem_raw) + 1023u) & ~1023u;
  unsigned char* gen = smem_raw + (base - tc::smem_u32(smem_raw));
  const uint32_t bar0 = base + SM::bar_off, bar1 = bar0 + 8;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(gen + SM::bar_off + 16);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int64_t row0 = (int64_t)blockIdx.x * BM;
  const int K = a.K1 + a.K2;
  const int nk = K / BK;
  const __nv_bfloat16* Bw = (const __nv_bfloat16*)a.B;

  if (tid == 0) {
    tc::mbar_init(bar0, 1);
    tc::mbar_init(bar1, 1);
    tc::fence_mbar_init();
  }
  if (warp == 0) tc::tmem_alloc<N>(tmem_slot);
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *tmem_slot;
  constexpr uint32_t IDESC = tc::idesc_bf16(128, N, 0, 0);

  for (int kc = 0; kc < nk; ++kc) {
    const int s = kc & 1;
    if (kc >= 2) tc::mbar_wait(s ? bar1 : bar0, (uint32_t)(((kc - 2) >> 1) & 1));  // MMAs of chunk kc-2 done
    const int k0 = kc * BK;
    // B slab: N rows x 128 B, 16-byte chunks via cp.async
#pragma unroll
    for (int i = 0; i < N * 8 / 256; ++i) {
      const int idx = tid + 256 * i;
      const int n = idx >> 3, ch = idx & 7;
      tc::cp_async16(base + SM::b_off(s) + tc::sw128_chunk_off(N, n, ch), Bw + (size_t)n * K + k0 + ch * 8);
    }
    tc::cp_async_commit();
    // A slab: 128 rows x 64 fp32 -> bf16
    const float* X = k0 < a.K1 ? a.X1 : a.X2;
    const int ld = k0 < a.K1 ? a.ld1 : a.ld2;
    const int kx = k0 < a.K1 ? k0 : k0 - a.K1;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int idx = tid + 256 * i;
      const int r = idx >> 4, c4 = idx & 15;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row0 + r < a.n) {
        v = *reinterpret_cast<const float4*>(X + (row0 + r) * ld + kx + c4 * 4);
        if (a.act_in) { v.x = silu_f(v.x); v.y = silu_f(v.y); v.z = silu_f(v.z); v.w = silu_f(v.w); }
      }
      uint2 pk;
      pk.x = tc::pack_bf16(v.x, v.y);
      pk.y = tc::pack_bf16(v.z, v.w);
      *reinterpret_cast<uint2*>(gen + SM::a_off(s) + tc::sw128_chunk_off(BM, r, c4 >> 1) + (c4 & 1) * 8) = pk;
    }
    tc::cp_async_wait<0>();
    tc::fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
      tc::fence_after_sync();
#pragma unroll
      for (int kk = 0; kk < BK / 16; ++kk) {
        const uint64_t ad = tc::smem_desc(base + SM::a_off(s) + kk * 32, 16, 1024, tc::LAYOUT_SW128);
        const uint64_t bd = tc::smem_desc(base + SM::b_off(s) + kk * 32, 16, 1024, tc::LAYOUT_SW128);
        tc::mma_bf16(tmem, ad, bd, IDESC, (kc | kk) != 0);
      }
      tc::mma_commit(s ? bar1 : bar0);
    }
  }
  {
    const int kl = nk - 1;
    tc::mbar_wait((kl & 1) ? bar1 : bar0, (uint32_t)((kl >> 1) & 1));
    tc::fence_after_sync();
  }

  // ---- epilogue: thread = (row, column half) ----
  const int q = warp & 3, hf = warp >> 2;
  const int64_t r = row0 + q * 32 + lane;
  const bool valid = r < a.n;
#pragma unroll 1
  for (int c0 = hf * (N / 2); c0 < (hf + 1) * (N / 2); c0 += 32) {
    float y[32];
    tc::tmem_ld32(tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)c0, y);
    if (valid) {
      if (a.bias) {
#pragma unroll
        for (int j = 0; j < 32; ++j) y[j] += __ldg(a.bias + c0 + j);
      }
      if (a.mul_dsilu) {
#pragma unroll
        for (int j = 0; j < 32; j += 4) {
          const float4 z = *reinterpret_cast<const float4*>(a.mul_dsilu + r * a.ldz + c0 + j);
          y[j] *= dsilu_f(z.x); y[j + 1] *= dsilu_f(z.y); y[j + 2] *= dsilu_f(z.z); y[j + 3] *= dsilu_f(z.w);
        }
      }
      if (a.residual) {
#pragma unroll
        for (int j = 0; j < 32; j += 4) {
          const float4 z = *reinterpret_cast<const float4*>(a.residual + r * a.ldr + c0 + j);
          y[j] += z.x; y[j + 1] += z.y; y[j + 2] += z.z; y[j + 3] += z.w;
        }
      }
      if (a.Y) {
#pragma unroll
        for (int j = 0; j < 32; j += 4)
          *reinterpret_cast<float4*>(a.Y + r * a.ldy + c0 + j) = make_float4(y[j], y[j + 1], y[j + 2], y[j + 3]);
      }
      if (a.Yh) {
#pragma unroll
        for (int j = 0; j < 32; j += 8) {
          uint4 pk;
          pk.x = tc::pack_f16(y[j], y[j + 1]); pk.y = tc::pack_f16(y[j + 2], y[j + 3]);
          pk.z = tc::pack_f16(y[j + 4], y[j + 5]); pk.w = tc::pack_f16(y[j + 6], y[j + 7]);
          *reinterpret_cast<uint4*>(a.Yh + r * a.ldy + c0 + j) = pk;
        }
      }
      if (a.Ybf) {
#pragma unroll
        for (int j = 0; j < 32; j += 8) {
          uint4 pk;
          pk.x = tc::pack_bf16(y[j], y[j + 1]); pk.y = tc::pack_bf16(y[j + 2], y[j + 3]);
          pk.z = tc::pack_bf16(y[j + 4], y[j + 5]); pk.w = tc::pack_bf16(y[j + 6], y[j + 7]);
          *reinterpret_cast<uint4*>(a.Ybf + r * a.ldy + c0 + j) = pk;
        }
      }
    }
  }
  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<N>(tmem);
}

template <int N>
int launch(mlip_ctx* ctx, const GemmArgs& a) {
  const size_t smem = NodeSmem<N>::bytes;
  MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_gemm_bf16<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_gemm_bf16<N><<<(unsigned)((a.n + BM - 1) / BM), 256, smem, ctx->stream>>>(a);
  ctx->launches++;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
}  // namespace

int mlip_gemm_bf16(mlip_ctx* ctx, const GemmArgs& a) {
  if (a.n <= 0) return MLIP_OK;
  if (a.K1 % BK || a.K2 % BK || a.K1 + a.K2 == 0) { ctx->set_error("gemm_bf16: K not a multiple of 64"); return MLIP_ERR_UNSUPPORTED; }
  if (a.N == 256) return launch<256>(ctx, a);
  if (a.N == 128) return launch<128>(ctx, a);
  ctx->set_error("gemm_bf16: N must be 128 or 256");
  return MLIP_ERR_UNSUPPORTED;
}
