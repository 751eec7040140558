// MLIP_FP32 node-level GEMMs on the tensor cores (steps A8, A9 and their adjoints at d = 128): the same 3-term bf16 split
// as the edge kernels (edge_x3.cu) for Y[n,N] = epi( act(X)[n,K] . B^T + bias ), X = [X1 | X2] fp32.
// One CTA computes a 128-row x 128-column output tile; K goes through shared memory in chunks of 64: all threads load the
// fp32 activations of the chunk (SiLU on load where asked), split them into three bf16 terms and write SWIZZLE_128B slabs,
// copy the pre-split weight chunk, and one elected lane issues 4 K steps x 6 MMAs. The main products a1 b1 and the five
// small terms go to separate fp32 accumulators in tensor memory (the tensor core truncates when it accumulates; the
// epilogue adds the two). Two CTAs per SM (96 KB of shared memory, 256 TMEM columns each): one converts while the other
// multiplies. The epilogue (bias, x SiLU'(Z), + residual) is the fp32 arithmetic of node_f32.cu.
// The node GEMMs of config 5 are 1-2 GFLOP each: on the CUDA cores they ran at a third of the FMA peak.
#include <cuda_bf16.h>
#include "common.cuh"
#include "mathfn.cuh"
#include "tc_images.cuh"
#include "tc_ptx.cuh"

namespace {
constexpr int BM = 128, BN = 128, BK = 64;
constexpr int NT = 256;
constexpr uint32_t SLAB = BM * BK * 2;   // one [128 x 64] bf16 SW128 slab = 16 KB

struct SMX {
  static constexpr uint32_t A = 0;                 // [3] slabs
  static constexpr uint32_t B = 3 * SLAB;          // [3] slabs
  static constexpr uint32_t bar = 6 * SLAB;        // one mbarrier
  static constexpr uint32_t slot = bar + 8;        // TMEM base address
  static constexpr uint32_t bytes = slot + 8 + 1024;   // + alignment slack
};

__device__ __forceinline__ void split3(float x0, float x1, uint32_t (&h)[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    h[i] = tc::pack_bf16(x0, x1);
    if (i < 2) { x0 -= tc::bf16_lo(h[i]); x1 -= tc::bf16_hi(h[i]); }
  }
}
__device__ __forceinline__ void tmem_ld16_raw(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
}

// 256-bit global accesses (32-byte aligned: activations come from the allocator, row strides are multiples of 64 floats).
// Plain (not .nc) loads: the residual may alias Y.
__device__ __forceinline__ void ld8(const float* p, float (&v)[8]) {
  asm volatile("ld.global.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
               : "l"(p)
               : "memory");
}
__device__ __forceinline__ void st8(float* p, const float (&v)[8]) {
  asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]),
               "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7])
               : "memory");
}

// Bx3: three split terms of B [N, K], each a K-major SWIZZLE_128B image with rows = N (tc_sw128_index)
__global__ void __launch_bounds__(NT, 2) k_gemm_x3(GemmArgs a, const __nv_bfloat16* __restrict__ Bx3) {
  extern __shared__ unsigned char smem_raw[];
  const uint32_t base = (tc::smem_u32(smem_raw) + 1023u) & ~1023u;
  unsigned char* gen = smem_raw + (base - tc::smem_u32(smem_raw));
  uint32_t* slot = reinterpret_cast<uint32_t*>(gen + SMX::slot);
  const uint32_t bar = base + SMX::bar;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int64_t row0 = (int64_t)blockIdx.x * BM;
  const int col0 = blockIdx.y * BN;
  const int K = a.K1 + a.K2, nk = K / BK;

  if (tid == 0) { tc::mbar_init(bar, 1); tc::fence_mbar_init(); }
  if (warp == 0) tc::tmem_alloc<2 * BN>(slot);
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *slot;
  const uint32_t TM = tmem, TS = tmem + BN;   // main / small-term accumulators
  constexpr uint32_t IDESC = tc::idesc_bf16(BM, BN, 0, 0);

  // loader mapping: 16 threads per row (4 consecutive k each), 16 rows per pass, 8 passes; the [128 x 64] chunk of the three
  // weight terms is 3 x 16 KB = 3072 x 16 B, 12 per thread. The global loads of chunk kb + 1 are issued right after the MMAs
  // of chunk kb, so their latency runs under those MMAs.
  const int c4 = tid & 15, r0 = tid >> 4;
  const uint4* Bsrc = reinterpret_cast<const uint4*>(Bx3);
  const size_t term = (size_t)a.N * K * 2 / 16;
  float4 v[8];
  uint4 w[12];
  auto load = [&](int kb) {
    const int k0 = kb * BK;
    const bool first = k0 < a.K1;
    const float* X = first ? a.X1 : a.X2;
    const int ld = first ? a.ld1 : a.ld2;
    const int kx = (first ? k0 : k0 - a.K1) + 4 * c4;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int64_t r = row0 + r0 + 16 * i;
      v[i] = r < a.n ? __ldg(reinterpret_cast<const float4*>(X + r * ld + kx)) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const size_t chunk = ((size_t)kb * a.N * BK + (size_t)col0 * BK) * 2 / 16;
#pragma unroll
    for (int j = 0; j < 12; ++j) {
      const int idx = tid + NT * j;          // 0..3071
      w[j] = __ldg(Bsrc + (idx >> 10) * term + chunk + (idx & 1023));
    }
  };
  uint32_t phase = 0;
  load(0);
  for (int kb = 0; kb < nk; ++kb) {
    if (kb > 0) {  // the MMAs of the previous chunk have read shared memory
      tc::mbar_wait_warp(bar, phase);
      phase ^= 1u;
    }
#pragma unroll
    for (int j = 0; j < 12; ++j) {
      const int idx = tid + NT * j;
      *reinterpret_cast<uint4*>(gen + SMX::B + (idx >> 10) * SLAB + (idx & 1023) * 16) = w[j];
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int r = r0 + 16 * i;
      float4 x = v[i];
      if (a.act_in) { x.x = silu_f(x.x); x.y = silu_f(x.y); x.z = silu_f(x.z); x.w = silu_f(x.w); }
      uint32_t h0[3], h1[3];
      split3(x.x, x.y, h0);
      split3(x.z, x.w, h1);
      // 8 bytes at element (r, 4 c4) of the slab: chunk (c4 / 2) ^ (r % 8), half c4 % 2
      const uint32_t off = (uint32_t)(r * 128 + (((c4 >> 1) ^ (r & 7)) << 4) + ((c4 & 1) << 3));
#pragma unroll
      for (int t = 0; t < 3; ++t) *reinterpret_cast<uint2*>(gen + SMX::A + t * SLAB + off) = make_uint2(h0[t], h1[t]);
    }
    tc::fence_proxy_async();
    __syncthreads();
    if (warp == 0) {
      tc::fence_after_sync();
      if (tc::elect_one()) {
        constexpr int IA[5] = {2, 1, 0, 1, 0}, IB[5] = {0, 1, 2, 0, 1};
#pragma unroll
        for (int kk = 0; kk < BK / 16; ++kk) {
          auto ad = [&](int t) { return tc::smem_desc(base + SMX::A + t * SLAB + kk * 32, 16, 1024, tc::LAYOUT_SW128); };
          auto bd = [&](int t) { return tc::smem_desc(base + SMX::B + t * SLAB + kk * 32, 16, 1024, tc::LAYOUT_SW128); };
#pragma unroll
          for (int t = 0; t < 5; ++t) tc::mma_bf16(TS, ad(IA[t]), bd(IB[t]), IDESC, (kb | kk | t) != 0);
          tc::mma_bf16(TM, ad(0), bd(0), IDESC, (kb | kk) != 0);
        }
        tc::mma_commit(bar);
      }
      __syncwarp();
    }
    if (kb + 1 < nk) load(kb + 1);
  }
  tc::mbar_wait_warp(bar, phase);
  tc::fence_after_sync();

  // ---- epilogue: thread = (row, 64 columns) ----
  const int row = (warp & 3) * 32 + lane, ch0 = (warp >> 2) * 64;
  const uint32_t tlane = (uint32_t)((warp & 3) * 32) << 16;
  const int64_t r = row0 + row;
#pragma unroll
  for (int cb = 0; cb < 4; ++cb) {
    uint32_t m[16], s[16];
    tmem_ld16_raw(TM + tlane + (uint32_t)(ch0 + 16 * cb), m);
    tmem_ld16_raw(TS + tlane + (uint32_t)(ch0 + 16 * cb), s);
    tc::tmem_wait_ld();
    if (r < a.n) {
      const int c = col0 + ch0 + 16 * cb;
      // 32 bytes (one sector) per access: the rows of a warp are ldy floats apart, so every access is its own sector anyway
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        float y[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) y[j] = __uint_as_float(m[8 * q + j]) + __uint_as_float(s[8 * q + j]);
        if (a.bias) {
          const float4 b0 = __ldg(reinterpret_cast<const float4*>(a.bias + c + 8 * q)), b1 = __ldg(reinterpret_cast<const float4*>(a.bias + c + 8 * q + 4));
          y[0] += b0.x; y[1] += b0.y; y[2] += b0.z; y[3] += b0.w; y[4] += b1.x; y[5] += b1.y; y[6] += b1.z; y[7] += b1.w;
        }
        if (a.mul_dsilu) {
          float z[8];
          ld8(a.mul_dsilu + r * a.ldz + c + 8 * q, z);
#pragma unroll
          for (int j = 0; j < 8; ++j) y[j] *= dsilu_f(z[j]);
        }
        if (a.residual) {
          float p[8];
          ld8(a.residual + r * a.ldr + c + 8 * q, p);
#pragma unroll
          for (int j = 0; j < 8; ++j) y[j] += p[j];
        }
        st8(a.Y + r * a.ldy + c + 8 * q, y);
      }
    }
  }
  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<2 * BN>(tmem);
}

__global__ void k_gemm_image_x3(const float* __restrict__ W, int N, int K, __nv_bfloat16* __restrict__ img) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * K) return;
  float x = W[idx];
  const int o = tc_sw128_index(N, idx / K, idx % K);
  for (int t = 0; t < 3; ++t) {
    const __nv_bfloat16 h = __float2bfloat16_rn(x);
    img[(size_t)t * N * K + o] = h;
    x -= __bfloat162float(h);
  }
}
}  // namespace

void mlip_make_gemm_image_x3(cudaStream_t st, const float* W, int N, int K, __nv_bfloat16* img) {
  k_gemm_image_x3<<<(N * K + 255) / 256, 256, 0, st>>>(W, N, K, img);
}

bool mlip_gemm_x3_supported(const GemmArgs& a) {
  return a.Y && !a.Ybf && !a.Yh && a.N % BN == 0 && a.K1 % BK == 0 && a.K2 % BK == 0 && a.K1 + a.K2 <= 256 && a.X1 && !a.X1b && !a.X2b;
}

int mlip_gemm_x3(mlip_ctx* ctx, const GemmArgs& a, const __nv_bfloat16* Bx3) {
  if (a.n <= 0) return MLIP_OK;
  dim3 grid((unsigned)((a.n + BM - 1) / BM), a.N / BN);
  MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_gemm_x3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMX::bytes));
  k_gemm_x3<<<grid, NT, SMX::bytes, ctx->stream>>>(a, Bx3);
  ctx->launches++;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
