// bf16 tensor-core node-level GEMM with fused prologue / epilogue (steps A8, A9 and their adjoints
// in the MLIP_BF16 path): Y[n,N] = epi( act(X)[n,K] . B^T + bias ), X = [X1 | X2] fp32 in global.
//
// The node GEMMs are HBM bound (fp32 activations in and out, 2 d^2 flop per 8..12 bytes per element),
// so the kernel is built to keep loads in flight, not to feed the tensor pipe: one persistent,
// warp-specialised CTA per SM walks over 128-row tiles;
//   warps 0..7   epilogue: TMEM -> registers -> per-warp 32x32 transpose through shared memory, so that
//                every global access of the epilogue (bias, SiLU' factor, residual, output) is a
//                full 128-byte row segment -> fp32 / f16 / bf16 rows
//   warp  8      one thread issues the tcgen05.mma (M=128, N, K=16) into one of TWO accumulators in
//                tensor memory, so the epilogue of tile t overlaps the main loop of tile t+1
//   warp  9      one thread streams the [N x 64] SWIZZLE_128B weight slabs (pre-built images, see
//                mlip_make_gemm_image) with cp.async.bulk
//   warps 10..17 activation producers: fp32 rows -> (SiLU) -> bf16 -> K-major SWIZZLE_128B slab, with
//                the loads of the next K chunk (also across tiles) in flight before the current one
//                is stored
// through a ring of STAGES (A slab | B slab) buffers guarded by full / empty mbarriers.
#include "common.cuh"
#include "mathfn.cuh"
#include "tc_images.cuh"
#include "tc_ptx.cuh"

namespace {
constexpr int BM = 128, BK = 64;
constexpr int N_EPI = 8, WARP_MMA = 8, WARP_B = 9, WARP_A0 = 10, N_AW = 8;
constexpr int N_THREADS = (WARP_A0 + N_AW) * 32;  // 576

template <int N>
struct NodeSmem {
  static constexpr int STAGES = N == 256 ? 4 : 6;
  static constexpr uint32_t a_bytes = BM * BK * 2;  // 16 KB
  static constexpr uint32_t b_bytes = N * BK * 2;   // 32 KB at N = 256
  static constexpr uint32_t stage_bytes = a_bytes + b_bytes;
  static constexpr uint32_t a_off(int s) { return s * stage_bytes; }
  static constexpr uint32_t b_off(int s) { return s * stage_bytes + a_bytes; }
  static constexpr uint32_t xpose = STAGES * stage_bytes;       // 8 warps x [32 x 32] fp32, chunk-swizzled
  static constexpr uint32_t bars = xpose + N_EPI * 4096;
  static constexpr uint32_t slot = bars + 8 * (2 * STAGES + 4);
  static constexpr uint32_t bytes = slot + 16 + 1024;           // + alignment slack
  static_assert(bytes <= 232448, "shared memory budget of one SM exceeded");
};

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ float4 ldg_stream_f4(const float* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}

__device__ __forceinline__ float4 ldg_f4(const float* p) {  // ordered with the stores of the same thread (residual may alias Y)
  float4 v;
  asm volatile("ld.global.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
  return v;
}

template <int N>
__global__ void __launch_bounds__(N_THREADS, 1) k_gemm_bf16(GemmArgs a, int64_t n_tiles) {
  extern __shared__ unsigned char smem_raw[];
  using SM = NodeSmem<N>;
  constexpr int STAGES = SM::STAGES;
  const uint32_t base = (tc::smem_u32(smem_raw) + 1023u) & ~1023u;  // SWIZZLE_128B slabs need 1024-byte alignment
  unsigned char* gen = smem_raw + (base - tc::smem_u32(smem_raw));
  auto full = [&](int s) -> uint32_t { return base + SM::bars + 8u * (uint32_t)s; };
  auto empty = [&](int s) -> uint32_t { return base + SM::bars + 8u * (uint32_t)(STAGES + s); };
  auto acc_full = [&](int b) -> uint32_t { return base + SM::bars + 8u * (uint32_t)(2 * STAGES + b); };
  auto acc_empty = [&](int b) -> uint32_t { return base + SM::bars + 8u * (uint32_t)(2 * STAGES + 2 + b); };
  uint32_t* slot = reinterpret_cast<uint32_t*>(gen + SM::slot);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int K = a.K1 + a.K2;
  const int nk = K / BK;
  const int64_t my_tiles = (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x;
  const int64_t total = my_tiles * nk;  // K chunks this CTA walks through

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { tc::mbar_init(full(s), N_AW + 1); tc::mbar_init(empty(s), 1); }
    for (int b = 0; b < 2; ++b) { tc::mbar_init(acc_full(b), 1); tc::mbar_init(acc_empty(b), N_EPI); }
    tc::fence_mbar_init();
  }
  if (warp == 0) tc::tmem_alloc<2 * N>(slot);
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *slot;

  if (warp >= WARP_A0) {
    // ======================= activation producers =======================
    const int pt = tid - WARP_A0 * 32;  // 0..255: thread = (16-byte column group c4, rows r0 + 16 i)
    const int c4 = pt & 15, r0 = pt >> 4;
    auto load = [&](float4 (&v)[8], int64_t g) {
      if (g >= total) return;
      const int64_t row0 = ((int64_t)blockIdx.x + (g / nk) * gridDim.x) * BM;
      const int k0 = (int)(g % nk) * BK;
      const float* X = k0 < a.K1 ? a.X1 : a.X2;
      const int ld = k0 < a.K1 ? a.ld1 : a.ld2;
      const int kx = (k0 < a.K1 ? k0 : k0 - a.K1) + c4 * 4;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int64_t r = row0 + r0 + 16 * i;
        v[i] = r < a.n ? ldg_stream_f4(X + r * ld + kx) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
    };
    auto store = [&](float4 (&v)[8], int64_t g) {
      if (g >= total) return;
      const int s = (int)(g % STAGES);
      tc::mbar_wait(empty(s), (uint32_t)(((g / STAGES) & 1) ^ 1));
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int r = r0 + 16 * i;
        float4 x = v[i];
        if (a.act_in) { x.x = silu_f(x.x); x.y = silu_f(x.y); x.z = silu_f(x.z); x.w = silu_f(x.w); }
        uint2 pk;
        pk.x = tc::pack_bf16(x.x, x.y);
        pk.y = tc::pack_bf16(x.z, x.w);
        *reinterpret_cast<uint2*>(gen + SM::a_off(s) + tc::sw128_chunk_off(BM, r, c4 >> 1) + (c4 & 1) * 8) = pk;
      }
      tc::fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(full(s));
    };
    float4 b0[8], b1[8];
    load(b0, 0);
    for (int64_t g = 0; g < total; g += 2) {
      load(b1, g + 1); store(b0, g);
      load(b0, g + 2); store(b1, g + 1);
    }
  } else if (warp == WARP_B) {
    // ======================= weight slab producer (one thread) =======================
    if (lane == 0) {
      const unsigned char* img = reinterpret_cast<const unsigned char*>(a.B);
      for (int64_t g = 0; g < total; ++g) {
        const int s = (int)(g % STAGES);
        tc::mbar_wait(empty(s), (uint32_t)(((g / STAGES) & 1) ^ 1));
        tc::mbar_expect_tx(full(s), SM::b_bytes);
        tc::bulk_g2s(base + SM::b_off(s), img + (size_t)(g % nk) * SM::b_bytes, SM::b_bytes, full(s));
      }
    }
  } else if (warp == WARP_MMA) {
    // ======================= MMA issuer (one thread) =======================
    if (lane == 0) {
      constexpr uint32_t IDESC = tc::idesc_bf16(128, N, 0, 0);
      int64_t g = 0;
      for (int64_t it = 0; it < my_tiles; ++it) {
        const int b = (int)(it & 1);
        tc::mbar_wait(acc_empty(b), (uint32_t)(((it >> 1) & 1) ^ 1));
        tc::fence_after_sync();
        for (int kc = 0; kc < nk; ++kc, ++g) {
          const int s = (int)(g % STAGES);
          tc::mbar_wait(full(s), (uint32_t)((g / STAGES) & 1));
          tc::fence_after_sync();
#pragma unroll
          for (int kk = 0; kk < BK / 16; ++kk)
            tc::mma_bf16(tmem + (uint32_t)(b * N), tc::smem_desc(base + SM::a_off(s) + kk * 32, 16, 1024, tc::LAYOUT_SW128),
                         tc::smem_desc(base + SM::b_off(s) + kk * 32, 16, 1024, tc::LAYOUT_SW128), IDESC, (kc | kk) != 0);
          tc::mma_commit(empty(s));
        }
        tc::mma_commit(acc_full(b));
      }
    }
  } else {
    // ======================= epilogue warps =======================
    const int q = warp & 3, hf = warp >> 2;
    float* xp = reinterpret_cast<float*>(gen + SM::xpose + warp * 4096);
    const int cj = lane & 7, rj = lane >> 3;  // after the transpose: thread = (row 4 i + rj, columns 4 cj .. 4 cj + 3)
    const float* zsrc = a.mul_dsilu ? a.mul_dsilu : a.residual;
    const int zld = a.mul_dsilu ? a.ldz : a.ldr;
    for (int64_t it = 0; it < my_tiles; ++it) {
      const int b = (int)(it & 1);
      const int64_t row0 = ((int64_t)blockIdx.x + it * gridDim.x) * BM + q * 32;
      tc::mbar_wait(acc_full(b), (uint32_t)((it >> 1) & 1));
      tc::fence_after_sync();
#pragma unroll 1
      for (int c0 = hf * (N / 2); c0 < (hf + 1) * (N / 2); c0 += 32) {
        uint32_t y[32];
        tc::tmem_ld32_nowait(tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(b * N + c0), y);
        const int c = c0 + 4 * cj;
        float4 bias = make_float4(0.f, 0.f, 0.f, 0.f);
        if (a.bias) bias = *reinterpret_cast<const float4*>(a.bias + c);
        // the epilogue operand (SiLU' argument or residual; no caller passes both) of the whole chunk is requested
        // before anything is stored, so the eight row segments cost one round trip, not eight
        float4 z[8];
        if (zsrc) {
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int64_t r = row0 + 4 * i + rj;
            z[i] = r < a.n ? ldg_f4(zsrc + r * zld + c) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
        }
        tc::tmem_wait_ld();
        __syncwarp();  // the previous chunk has been read out of the staging tile
#pragma unroll
        for (int j = 0; j < 8; ++j)
          *reinterpret_cast<uint4*>(xp + lane * 32 + ((j ^ (lane & 7)) << 2)) = make_uint4(y[4 * j], y[4 * j + 1], y[4 * j + 2], y[4 * j + 3]);
        __syncwarp();
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int rl = 4 * i + rj;
          const int64_t r = row0 + rl;
          float4 v = *reinterpret_cast<const float4*>(xp + rl * 32 + ((cj ^ (rl & 7)) << 2));
          if (r < a.n) {
            v.x += bias.x; v.y += bias.y; v.z += bias.z; v.w += bias.w;
            if (a.mul_dsilu) {
              v.x *= dsilu_f(z[i].x); v.y *= dsilu_f(z[i].y); v.z *= dsilu_f(z[i].z); v.w *= dsilu_f(z[i].w);
            } else if (a.residual) {
              v.x += z[i].x; v.y += z[i].y; v.z += z[i].z; v.w += z[i].w;
            }
            if (a.Y) *reinterpret_cast<float4*>(a.Y + r * a.ldy + c) = v;
            if (a.Yh) *reinterpret_cast<uint2*>(a.Yh + r * a.ldy + c) = make_uint2(tc::pack_f16(v.x, v.y), tc::pack_f16(v.z, v.w));
            if (a.Ybf) *reinterpret_cast<uint2*>(a.Ybf + r * a.ldy + c) = make_uint2(tc::pack_bf16(v.x, v.y), tc::pack_bf16(v.z, v.w));
          }
        }
      }
      tc::fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(acc_empty(b));
    }
  }

  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<2 * N>(tmem);
}

// W [N, K] fp32 row-major -> scale * W as the bf16 SWIZZLE_128B K-major operand image the kernel streams:
// K/64 slabs of [N x 64] (N * 128 bytes each), element (n, k) at tc_sw128_index(N, n, k)
__global__ void k_gemm_image(const float* __restrict__ W, int N, int K, float scale, __nv_bfloat16* __restrict__ img) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * K) return;
  const int n = idx / K, k = idx % K;
  img[tc_sw128_index(N, n, k)] = __float2bfloat16_rn(scale * W[idx]);
}

template <int N>
int launch(mlip_ctx* ctx, const GemmArgs& a) {
  const size_t smem = NodeSmem<N>::bytes;
  static bool configured = false;
  if (!configured) {
    MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_gemm_bf16<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = true;
  }
  const int64_t tiles = (a.n + BM - 1) / BM;
  const unsigned grid = (unsigned)(tiles < ctx->num_sms ? tiles : ctx->num_sms);
  k_gemm_bf16<N><<<grid, N_THREADS, smem, ctx->stream>>>(a, tiles);
  ctx->launches++;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
}  // namespace

void mlip_make_gemm_image(cudaStream_t st, const float* W, int N, int K, float scale, __nv_bfloat16* img) {
  k_gemm_image<<<(N * K + 255) / 256, 256, 0, st>>>(W, N, K, scale, img);
}

int mlip_gemm_bf16(mlip_ctx* ctx, const GemmArgs& a) {
  if (a.n <= 0) return MLIP_OK;
  if (a.K1 % BK || a.K2 % BK || a.K1 + a.K2 == 0) { ctx->set_error("gemm_bf16: K not a multiple of 64"); return MLIP_ERR_UNSUPPORTED; }
  if (a.mul_dsilu && a.residual) { ctx->set_error("gemm_bf16: SiLU' factor and residual in one epilogue are not supported"); return MLIP_ERR_UNSUPPORTED; }
  if (a.N == 256) return launch<256>(ctx, a);
  if (a.N == 128) return launch<128>(ctx, a);
  ctx->set_error("gemm_bf16: N must be 128 or 256");
  return MLIP_ERR_UNSUPPORTED;
}
