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

// RES: the whole weight image (K <= RES_K) stays resident in shared memory for the life of the CTA and only the
// activation slabs go through the ring. Re-streaming the [N x K] image from L2 for every 128-row tile costs as many
// bytes over the L2 -> SM fabric as the activations themselves (148 SMs x 128 KB per tile), and that fabric, not HBM,
// is what the streaming form saturates. K = 2d (two column blocks) does not fit and keeps the streaming ring.
template <int N, bool RES>
struct NodeSmem {
  static constexpr int STAGES = RES ? 4 : (N == 256 ? 4 : 6);
  static constexpr uint32_t a_bytes = BM * BK * 2;  // 16 KB
  static constexpr uint32_t b_bytes = N * BK * 2;   // 32 KB at N = 256
  static constexpr int RES_K = 256;                 // resident image: up to [N x 256] bf16 (128 KB at N = 256)
  static constexpr uint32_t stage_bytes = RES ? a_bytes : a_bytes + b_bytes;
  static constexpr uint32_t a_off(int s) { return s * stage_bytes; }
  static constexpr uint32_t b_off(int s) { return s * stage_bytes + a_bytes; }     // streaming form
  static constexpr uint32_t b_res = STAGES * stage_bytes;                          // resident form: K/64 slabs
  static constexpr uint32_t xpose = STAGES * stage_bytes + (RES ? (RES_K / BK) * b_bytes : 0);  // 8 warps x [32 x 32] fp32
  static constexpr uint32_t bars = xpose + N_EPI * 4096;
  static constexpr uint32_t slot = bars + 8 * (2 * STAGES + 5);
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

// ZM: epilogue operand (0 none, 1 y *= SiLU'(Z), 2 y += R); OM: outputs (bit 0 fp32 Y, bit 1 f16 Yh, bit 2 bf16 Ybf) --
// compile-time, so that the read-out loop is straight-line code
// RAW: every column block is bf16 (X1b / X2b): the producers only copy, 16 bytes per thread and row, and keep FOUR K
// chunks (one whole 128 x 256 tile) in flight in the registers that hold two fp32 chunks otherwise -- the node GEMMs are
// bound by the latency of these loads (about 2.5 us under load), not by their bytes
template <int N, int ZM, int OM, bool RES, bool RAW>
__global__ void __launch_bounds__(N_THREADS, 1) k_gemm_bf16(GemmArgs a, int n_tiles) {
  extern __shared__ unsigned char smem_raw[];
  using SM = NodeSmem<N, RES>;
  constexpr int STAGES = SM::STAGES;
  const uint32_t base = (tc::smem_u32(smem_raw) + 1023u) & ~1023u;  // SWIZZLE_128B slabs need 1024-byte alignment
  unsigned char* gen = smem_raw + (base - tc::smem_u32(smem_raw));
  auto full = [&](int s) -> uint32_t { return base + SM::bars + 8u * (uint32_t)s; };
  auto empty = [&](int s) -> uint32_t { return base + SM::bars + 8u * (uint32_t)(STAGES + s); };
  auto acc_full = [&](int b) -> uint32_t { return base + SM::bars + 8u * (uint32_t)(2 * STAGES + b); };
  auto acc_empty = [&](int b) -> uint32_t { return base + SM::bars + 8u * (uint32_t)(2 * STAGES + 2 + b); };
  const uint32_t w_full = base + SM::bars + 8u * (uint32_t)(2 * STAGES + 4);  // resident weight image has landed
  uint32_t* slot = reinterpret_cast<uint32_t*>(gen + SM::slot);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int K = a.K1 + a.K2;
  const int nk = K / BK;
  const int my_tiles = (n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total = my_tiles * nk;  // K chunks this CTA walks through (32-bit index arithmetic throughout)

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { tc::mbar_init(full(s), RES ? N_AW : N_AW + 1); tc::mbar_init(empty(s), 1); }
    tc::mbar_init(w_full, 1);
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
    // a chunk comes from X1 / X2 as fp32 (converted here) or from X1b / X2b as bf16 (copied: 8 bytes per thread and row,
    // carried in the first two lanes of the float4)
    auto load = [&](float4 (&v)[8], int g) {
      if (g >= total) return;
      const int64_t row0 = ((int64_t)blockIdx.x + (int64_t)(g / nk) * gridDim.x) * BM;
      const int k0 = (g % nk) * BK;
      const bool first = k0 < a.K1;
      const int ld = first ? a.ld1 : a.ld2;
      const int kx = (first ? k0 : k0 - a.K1) + c4 * 4;
      const mlip_nodeop* Xb = first ? a.X1b : a.X2b;
      if (Xb) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int64_t r = row0 + r0 + 16 * i;
          uint2 u = make_uint2(0u, 0u);
          if (r < a.n) asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(u.x), "=r"(u.y) : "l"(Xb + r * ld + kx));
          v[i] = make_float4(__uint_as_float(u.x), __uint_as_float(u.y), 0.f, 0.f);
        }
      } else {
        const float* X = first ? a.X1 : a.X2;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int64_t r = row0 + r0 + 16 * i;
          v[i] = r < a.n ? ldg_stream_f4(X + r * ld + kx) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
    };
    auto store = [&](float4 (&v)[8], int g) {
      if (g >= total) return;
      const int s = g % STAGES;
      const bool raw = ((g % nk) * BK < a.K1 ? a.X1b : a.X2b) != nullptr;
      tc::mbar_wait_warp(empty(s), (uint32_t)(((g / STAGES) & 1) ^ 1));
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int r = r0 + 16 * i;
        float4 x = v[i];
        uint2 pk;
        if (raw) {
          pk = make_uint2(__float_as_uint(x.x), __float_as_uint(x.y));
        } else {
          if (a.act_in) { x.x = silu_f(x.x); x.y = silu_f(x.y); x.z = silu_f(x.z); x.w = silu_f(x.w); }
          pk.x = tc::pack_op(x.x, x.y);
          pk.y = tc::pack_op(x.z, x.w);
        }
        *reinterpret_cast<uint2*>(gen + SM::a_off(s) + tc::sw128_chunk_off(BM, r, c4 >> 1) + (c4 & 1) * 8) = pk;
      }
      tc::fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(full(s));
    };
    if constexpr (RAW) {
      const int c8 = pt & 7, rr = pt >> 3;  // thread = (16-byte chunk of the 128-byte slab row, rows rr + 32 i)
      auto rload = [&](uint4 (&v)[4], int g) {
        if (g >= total) return;
        const int64_t row0 = ((int64_t)blockIdx.x + (int64_t)(g / nk) * gridDim.x) * BM;
        const int k0 = (g % nk) * BK;
        const bool first = k0 < a.K1;
        const mlip_nodeop* Xb = (first ? a.X1b : a.X2b) + (first ? k0 : k0 - a.K1) + c8 * 8;
        const int ld = first ? a.ld1 : a.ld2;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int64_t r = row0 + rr + 32 * i;
          v[i] = make_uint4(0u, 0u, 0u, 0u);
          if (r < a.n)
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(v[i].x), "=r"(v[i].y), "=r"(v[i].z), "=r"(v[i].w) : "l"(Xb + r * ld));
        }
      };
      auto rstore = [&](uint4 (&v)[4], int g) {
        if (g >= total) return;
        const int s = g % STAGES;
        tc::mbar_wait_warp(empty(s), (uint32_t)(((g / STAGES) & 1) ^ 1));
#pragma unroll
        for (int i = 0; i < 4; ++i)
          *reinterpret_cast<uint4*>(gen + SM::a_off(s) + tc::sw128_chunk_off(BM, rr + 32 * i, c8)) = v[i];
        tc::fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive(full(s));
      };
      uint4 r0b[4], r1b[4], r2b[4], r3b[4];
      rload(r0b, 0); rload(r1b, 1); rload(r2b, 2);
      for (int g = 0; g < total; g += 4) {
        rload(r3b, g + 3); rstore(r0b, g);
        rload(r0b, g + 4); rstore(r1b, g + 1);
        rload(r1b, g + 5); rstore(r2b, g + 2);
        rload(r2b, g + 6); rstore(r3b, g + 3);
      }
    } else {
      float4 b0[8], b1[8];
      load(b0, 0);
      for (int g = 0; g < total; g += 2) {
        load(b1, g + 1); store(b0, g);
        load(b0, g + 2); store(b1, g + 1);
      }
    }
  } else if (warp == WARP_B) {
    // ======================= weight slab producer (one thread) =======================
    if (lane == 0) {
      const unsigned char* img = reinterpret_cast<const unsigned char*>(a.B);
      if (RES) {
        tc::mbar_expect_tx(w_full, (uint32_t)nk * SM::b_bytes);
        for (int kc = 0; kc < nk; ++kc)
          tc::bulk_g2s(base + SM::b_res + (uint32_t)kc * SM::b_bytes, img + (size_t)kc * SM::b_bytes, SM::b_bytes, w_full);
      }
      for (int g = 0; !RES && g < total; ++g) {
        const int s = g % STAGES;
        tc::mbar_wait(empty(s), (uint32_t)(((g / STAGES) & 1) ^ 1));
        tc::mbar_expect_tx(full(s), SM::b_bytes);
        tc::bulk_g2s(base + SM::b_off(s), img + (size_t)(g % nk) * SM::b_bytes, SM::b_bytes, full(s));
      }
    }
  } else if (warp == WARP_MMA) {
    // ======================= MMA issuer (one thread) =======================
    if (lane == 0) {
      constexpr uint32_t IDESC = tc::idesc_op(128, N, 0, 0);
      int g = 0;
      if (RES) tc::mbar_wait(w_full, 0u);
      for (int it = 0; it < my_tiles; ++it) {
        const int b = it & 1;
        tc::mbar_wait(acc_empty(b), (uint32_t)(((it >> 1) & 1) ^ 1));
        tc::fence_after_sync();
        for (int kc = 0; kc < nk; ++kc, ++g) {
          const int s = g % STAGES;
          tc::mbar_wait(full(s), (uint32_t)((g / STAGES) & 1));
          tc::fence_after_sync();
#pragma unroll
          for (int kk = 0; kk < BK / 16; ++kk)
            tc::mma_bf16(tmem + (uint32_t)(b * N), tc::smem_desc(base + SM::a_off(s) + kk * 32, 16, 1024, tc::LAYOUT_SW128),
                         tc::smem_desc(base + (RES ? SM::b_res + (uint32_t)kc * SM::b_bytes : SM::b_off(s)) + kk * 32, 16, 1024,
                                       tc::LAYOUT_SW128),
                         IDESC, (kc | kk) != 0);
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
    const float* zsrc = ZM == 1 ? a.mul_dsilu : a.residual;
    const int zld = ZM == 1 ? a.ldz : a.ldr;
    constexpr int NC = N / 64;  // 32-column chunks per warp
    for (int it = 0; it < my_tiles; ++it) {
      const int b = it & 1;
      const int64_t row0 = ((int64_t)blockIdx.x + (int64_t)it * gridDim.x) * BM + q * 32;
      const bool all_rows = row0 + 32 <= a.n;
      tc::mbar_wait_warp(acc_full(b), (uint32_t)((it >> 1) & 1));
      tc::fence_after_sync();
#pragma unroll
      for (int k = 0; k < NC; ++k) {
        const int c0 = hf * (N / 2) + 32 * k;
        uint32_t y[32];
        tc::tmem_ld32_nowait(tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)(b * N + c0), y);
        const int c = c0 + 4 * cj;
        float4 bias = make_float4(0.f, 0.f, 0.f, 0.f);
        if (a.bias) bias = *reinterpret_cast<const float4*>(a.bias + c);
        // the epilogue operand (SiLU' argument or residual) of the whole chunk is requested before anything is stored, so
        // the eight row segments cost one round trip (under the accumulator read-out and the staging), not eight
        float4 z[8];
        if (ZM != 0) {
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int64_t r = row0 + 4 * i + rj;
            z[i] = (all_rows || r < a.n) ? ldg_f4(zsrc + r * zld + c) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
        }
        tc::tmem_wait_ld();
        __syncwarp();  // the previous chunk has been read out of the staging tile
#pragma unroll
        for (int j = 0; j < 8; ++j)
          *reinterpret_cast<uint4*>(xp + lane * 32 + ((j ^ (lane & 7)) << 2)) = make_uint4(y[4 * j], y[4 * j + 1], y[4 * j + 2], y[4 * j + 3]);
        __syncwarp();
        float4 v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int rl = 4 * i + rj;
          v[i] = *reinterpret_cast<const float4*>(xp + rl * 32 + ((cj ^ (rl & 7)) << 2));
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int64_t r = row0 + 4 * i + rj;
          const bool ok = all_rows || r < a.n;
          float4 w = v[i];
          w.x += bias.x; w.y += bias.y; w.z += bias.z; w.w += bias.w;
          if (ZM == 1) { w.x *= dsilu_f(z[i].x); w.y *= dsilu_f(z[i].y); w.z *= dsilu_f(z[i].z); w.w *= dsilu_f(z[i].w); }
          if (ZM == 2) { w.x += z[i].x; w.y += z[i].y; w.z += z[i].z; w.w += z[i].w; }
          if (ok) {
            if (OM & 1) *reinterpret_cast<float4*>(a.Y + r * a.ldy + c) = w;
            if (OM & 2) *reinterpret_cast<uint2*>(a.Yh + r * a.ldy + c) = make_uint2(tc::pack_f16(w.x, w.y), tc::pack_f16(w.z, w.w));
            if (OM & 4) *reinterpret_cast<uint2*>(a.Ybf + r * a.ldy + c) = make_uint2(tc::pack_op(w.x, w.y), tc::pack_op(w.z, w.w));
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
__global__ void k_gemm_image(const float* __restrict__ W, int N, int K, float scale, mlip_nodeop* __restrict__ img) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * K) return;
  const int n = idx / K, k = idx % K;
  img[tc_sw128_index(N, n, k)] = tc::float_to_op(scale * W[idx]);
}

template <int N, int ZM, int OM, bool RES, bool RAW>
int launch_raw(mlip_ctx* ctx, const GemmArgs& a) {
  const size_t smem = NodeSmem<N, RES>::bytes;
  static bool configured = false;
  if (!configured) {
    MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_gemm_bf16<N, ZM, OM, RES, RAW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = true;
  }
  const int64_t tiles = (a.n + BM - 1) / BM;
  const unsigned grid = (unsigned)(tiles < ctx->num_sms ? tiles : ctx->num_sms);
  k_gemm_bf16<N, ZM, OM, RES, RAW><<<grid, N_THREADS, smem, ctx->stream>>>(a, (int)tiles);
  ctx->launches++;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
template <int N, int ZM, int OM, bool RES>
int launch_res(mlip_ctx* ctx, const GemmArgs& a) {
  const bool raw = (a.K1 == 0 || a.X1b) && (a.K2 == 0 || a.X2b) && !a.act_in;
  return raw ? launch_raw<N, ZM, OM, RES, true>(ctx, a) : launch_raw<N, ZM, OM, RES, false>(ctx, a);
}
template <int N, int ZM, int OM>
int launch_one(mlip_ctx* ctx, const GemmArgs& a) {
  if (a.K1 + a.K2 <= NodeSmem<N, true>::RES_K) return launch_res<N, ZM, OM, true>(ctx, a);
  return launch_res<N, ZM, OM, false>(ctx, a);
}
template <int N, int ZM>
int launch_z(mlip_ctx* ctx, const GemmArgs& a) {
  const int om = (a.Y ? 1 : 0) | (a.Yh ? 2 : 0) | (a.Ybf ? 4 : 0);
  switch (om) {
    case 1: return launch_one<N, ZM, 1>(ctx, a);
    case 2: return launch_one<N, ZM, 2>(ctx, a);
    case 4: return launch_one<N, ZM, 4>(ctx, a);
    case 5: return launch_one<N, ZM, 5>(ctx, a);
    default: ctx->set_error("gemm_bf16: output set must be fp32, f16, bf16 or fp32 + bf16"); return MLIP_ERR_UNSUPPORTED;
  }
}
template <int N>
int launch(mlip_ctx* ctx, const GemmArgs& a) {
  if (a.mul_dsilu) return launch_z<N, 1>(ctx, a);
  if (a.residual) return launch_z<N, 2>(ctx, a);
  return launch_z<N, 0>(ctx, a);
}
}  // namespace

void mlip_make_gemm_image(cudaStream_t st, const float* W, int N, int K, float scale, mlip_nodeop* img) {
  k_gemm_image<<<(N * K + 255) / 256, 256, 0, st>>>(W, N, K, scale, img);
}

int mlip_gemm_bf16(mlip_ctx* ctx, const GemmArgs& a) {
  if (a.n <= 0) return MLIP_OK;
  if (a.K1 % BK || a.K2 % BK || a.K1 + a.K2 == 0) { ctx->set_error("gemm_bf16: K not a multiple of 64"); return MLIP_ERR_UNSUPPORTED; }
  if ((a.X1b && a.X1) || (a.X2b && a.X2) || ((a.X1b || a.X2b) && a.act_in)) {
    ctx->set_error("gemm_bf16: a column block is either fp32 or bf16; SiLU on load needs fp32");
    return MLIP_ERR_INVALID_ARG;
  }
  if (a.mul_dsilu && a.residual) { ctx->set_error("gemm_bf16: SiLU' factor and residual in one epilogue are not supported"); return MLIP_ERR_UNSUPPORTED; }
  if ((a.n + BM - 1) / BM >= (int64_t)1 << 24) { ctx->set_error("gemm_bf16: too many rows"); return MLIP_ERR_OVERFLOW; }
  if (a.N == 256) return launch<256>(ctx, a);
  if (a.N == 128) return launch<128>(ctx, a);
  ctx->set_error("gemm_bf16: N must be 128 or 256");
  return MLIP_ERR_UNSUPPORTED;
}
