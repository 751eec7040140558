// MLIP_FP32 path of the fused edge kernels (A6, A7, edge part of A10) on the tensor cores, d = 128: every
// contraction runs on tcgen05 with fp32 operands SPLIT INTO THREE bf16 TERMS, x = x1 + x2 + x3 with
// x1 = bf16(x), x2 = bf16(x - x1), x3 = bf16(x - x1 - x2) (24 significant bits, the exponent range of fp32: no
// range contract as in the MLIP_BF16 path). A product a b is evaluated as the six terms a1 b1 + a1 b2 + a2 b1 +
// a1 b3 + a2 b2 + a3 b1 accumulated in fp32 in tensor memory; what is dropped is below 2^-24 |a b|. Six bf16 MMAs
// at 8192 flop/clk/SM replace fp32 FMAs at 256 flop/clk/SM. Everything between the contractions (gathers, SiLU,
// envelope, radial basis) is fp32 arithmetic (MUFU ex2 / rcp approximations of 1-2 ulp, as in edge_f32.cu).
//
// One persistent CTA per SM walks over tiles of 128 receiver-sorted edges; the split images of W2 [d,d] and of
// [W1c | W3] [d,32] stay in shared memory (120 KB), one set of split operand slabs (96 KB) is rewritten per phase.
//   warps 0..15  epilogue: thread = (edge row, 8 channels per step, 4 steps); TMEM -> registers -> fp32 arithmetic -> three
//                bf16 terms -> SW128 slabs. A step completes TWO K steps of the MMAs (16 channels each, 8 warps each), so
//                the tensor core trails the epilogue by a quarter of a phase instead of half of it
//   warp 16      MMA issuer: the whole warp follows the barriers, one ELECTED lane issues (tc::elect_one: a divergent
//                `if (lane == 0)` costs 60 cycles per MMA in uniformisation loops, measured)
//   warp 17      segment analysis of the tile: receivers in order of appearance, destinations, 0/1 selector
// Per tile:
//   P0  envelope, radial basis; A0 = [e_hat | t_e] [128,32] in three terms. Computed in registers under the last MMAs
//       of the previous tile and stored as soon as they are done (A0 aliases the slabs).
//   G1  X = A0 . [W1c | W3]^T                               (K = 32; t_e = 0 without the three-body term)
//   E1  a = X + P_i + Q_j ; s = SiLU(a) -> slabs ; the reverse pass keeps SiLU'(a) in registers
//   G2  Y = s . W2^T
//   E2  forward : phi = alpha u_e SiLU(Y + b2) -> slabs
//       reverse : pbar = alpha u_e mbar_i SiLU'(p) -> slabs ; ubar_e = alpha <mbar_i, phi_e>
//   G3  X = pbar . W2           (reverse; the same W2 images read MN-major)
//   E3  abar = X SiLU'(a) -> slabs, and -> global spill (fp32, read back through rev[] by k_gather_rev_f32) AFTER the
//       last slab is published: the proxy fence of a publication waits for global stores issued before it (measured)
//   G4  [ebar | tbar] = abar . [W1c | W3]   (N = 32, the G1 images read MN-major)
//   GS  segmented sum over runs of equal receiver as an MMA with the 0/1 selector (three terms: the selector is
//       exact): Yseg[channel, r] = slab^T . Sel ; m_i (forward) / Pbar_i (reverse). Tiles with more than 16
//       receivers sum the slabs in a shared-memory loop.
//   E4  rbar_e += ubar_e u' + sum_k ebar_k (u' g_k + u g'_k) ; tbar_e -> global. E4 and the read-out of Yseg are
//       deferred until A0 of the next tile is published, so they run under its G1.
// All row gathers (P_i, Q_j, mbar_i, t_e) and the spill use 256-bit accesses: the rows of a tile are 512 bytes apart,
// every lane costs an L1 tag cycle per instruction. Segments that straddle tiles go through per-tile head / tail rows
// and a fix-up kernel, as in edge_f32.cu. The only reduction instruction is the one addition per edge and launch into
// rbar (order fixed by the launch order): results are bitwise reproducible.
#include <cuda_bf16.h>
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"
#include "tc_images.cuh"
#include "tc_ptx.cuh"

namespace {
constexpr int D = 128;            // channels (the only width this kernel is built for)
constexpr int TE = 128;           // edges per tile = MMA M
constexpr int N_EPI_WARPS = 16;   // epilogue warp = (lane quarter q = warp % 4, column group g = warp / 4)
constexpr int MMA_WARP = 16;      // one elected lane issues every MMA
constexpr int SEG_WARP = 17;      // segment analysis of the tile, ahead of its read-out
constexpr int NT = 18 * 32;
constexpr int NCH = D / 64;       // 64-channel operand slabs
constexpr int K1 = 32;            // K of G1: 16 radial + 16 angle terms
constexpr int SLAB = TE * 128;    // one [128 x 64] bf16 SW128 slab
constexpr int MAX_SEG = 16;       // receivers per tile handled by the selector MMA

struct Seg {
  float* dst[MAX_SEG];
  int R;
  int pad[3];
};

struct SM {  // shared-memory carve-up, byte offsets from the (1024-byte aligned) base
  static constexpr uint32_t w2 = 0;                               // [3][D x D] bf16, K-major SW128
  static constexpr uint32_t w13 = w2 + 3 * D * D * 2;             // [3][D x 32] bf16, K-major no swizzle
  static constexpr uint32_t A = w13 + 3 * D * K1 * 2;             // [3][NCH] slabs; A0 [3][128 x 32] aliases the start
  static constexpr uint32_t sel = A + 3 * NCH * SLAB;             // [16 x 128] bf16, K-major no swizzle
  static constexpr uint32_t recv = sel + MAX_SEG * TE * 2;        // int[128] receivers (fallback of the segmented sum)
  static constexpr uint32_t w = recv + TE * 4;                    // float[128] alpha u_e
  static constexpr uint32_t ubar = w + TE * 4;                    // float[4][128]
  static constexpr uint32_t seg = ubar + 4 * TE * 4;              // Seg
  static constexpr uint32_t bar = seg + sizeof(Seg);              // mbarriers
  static constexpr uint32_t slot = bar + 16 * 8;                  // TMEM base address
  static constexpr uint32_t bytes = slot + 8;
  static_assert(bytes <= 232448 - 1024, "shared memory budget of one SM exceeded");
};
// Tensor memory. The tensor core adds into its fp32 accumulator with truncation (round toward zero): a chain of n accumulations
// shrinks the result by about n / 2 ulp, systematically -- 48 accumulations per GEMM (8 K steps x 6 terms) put 4e-6 on the
// energy of a dense system (196 neighbours; measured against the float64 reference of the tests), beyond the 1e-5 per-atom bound in places. So every
// GEMM has TWO accumulators: the main one takes the 8 products a1 b1 of its K steps only, the other the five small terms,
// whose truncation errors are 2^-8 smaller; the epilogue adds the two in fp32 (round to nearest).
//   X [0,128) | Xs [128,256) | Y [256,384) | Ys [384,512); the outputs of GS and G4 (16 + 16 and 32 + 32 columns) alias the
//   head of Y, which is dead by then (the MMA warp waits for the read-out of tile t before G2 of tile t + 1 overwrites Y)
constexpr int TMEM_COLS = 512;
// B_S + k: the 16 channels 16 k .. 16 k + 15 (= K step k of the MMAs, slab k / 4) of an operand are written by the eight
// warps of column groups 2 (k % 2), 2 (k % 2) + 1 in step k / 2
enum { B_A0 = 0, B_S = 1 /* .. + 4 NCH */, B_G1 = 1 + 4 * NCH, B_G2, B_G3, B_FIN, B_SEG, B_RO, N_BARS };
static_assert(N_BARS <= 16, "barrier area");

__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// x = h[0] + h[1] + h[2] (bf16 each), two values per register
__device__ __forceinline__ void split3(float x0, float x1, uint32_t (&h)[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    h[i] = tc::pack_bf16(x0, x1);
    if (i < 2) { x0 -= tc::bf16_lo(h[i]); x1 -= tc::bf16_hi(h[i]); }
  }
}
constexpr int CPS = 8;            // channels per thread and step (see kst() below). Measured on config 5, reverse kernel: CPS = 16
                                  // (one K step per column group) 28.0 ms, CPS = 8 25.4 ms, CPS = 4 31.6 ms (twice the loads, stores and fences)
// N (4 or 8) consecutive channels of one row -> 2 N bytes in each of the three split slabs
template <int N>
__device__ __forceinline__ void store_split(unsigned char* A, uint32_t off, const float (&v)[N]) {
  uint32_t p[3][N / 2];
#pragma unroll
  for (int j = 0; j < N / 2; ++j) {
    uint32_t h[3];
    split3(v[2 * j], v[2 * j + 1], h);
    p[0][j] = h[0]; p[1][j] = h[1]; p[2][j] = h[2];
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    if constexpr (N == 8) *reinterpret_cast<uint4*>(A + i * (NCH * SLAB) + off) = make_uint4(p[i][0], p[i][1], p[i][2], p[i][3]);
    else *reinterpret_cast<uint2*>(A + i * (NCH * SLAB) + off) = make_uint2(p[i][0], p[i][1]);
  }
}
template <int N>
__device__ __forceinline__ void tmem_ld_raw(uint32_t taddr, uint32_t (&r)[N]) {
  static_assert(N == 4 || N == 8 || N == 16, "columns per load");
  if constexpr (N == 16)
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
  else if constexpr (N == 8)
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
  else
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(taddr)
                 : "memory");
}
// v = main accumulator + accumulator of the small terms (N columns of this thread's row), added in fp32
template <int N>
__device__ __forceinline__ void tmem_ld_sum(uint32_t t_main, uint32_t t_small, float (&v)[N]) {
  uint32_t a[N], b[N];
  tmem_ld_raw<N>(t_main, a);
  tmem_ld_raw<N>(t_small, b);
  tc::tmem_wait_ld();
#pragma unroll
  for (int i = 0; i < N; ++i) v[i] = __uint_as_float(a[i]) + __uint_as_float(b[i]);
}
// SiLU and its derivative in seven instructions: sigma = rcp(1 + ex2(-x log2 e)) with the two MUFU approximations (2 ulp /
// 1 ulp, flush-to-zero: no denormal fix-up code), y = x sigma, y' = sigma + y (1 - sigma). x -> -inf gives ex2 = inf, sigma = 0.
__device__ __forceinline__ float sigmoid_x3(float x) {
  float t, sg;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(t) : "f"(-1.4426950408889634f * x));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(sg) : "f"(1.0f + t));
  return sg;
}
__device__ __forceinline__ float silu_x3(float x) { return x * sigmoid_x3(x); }
__device__ __forceinline__ void silu_both_x3(float x, float& y, float& dy) {
  const float sg = sigmoid_x3(x);
  y = x * sg;
  dy = fmaf(y, 1.0f - sg, sg);
}
// Gaussian radial basis g_k(r) = exp(-gamma (r - k Delta)^2) with the constants hoisted out of the per-edge code
struct Rbf {
  float delta, neg_gamma_l2e, two_gamma;
  __device__ __forceinline__ Rbf(float r_cut, int n_rbf) {
    delta = r_cut / (float)(n_rbf - 1);
    const float gamma = 0.5f / (delta * delta);
    neg_gamma_l2e = -1.4426950408889634f * gamma;
    two_gamma = 2.0f * gamma;
  }
  __device__ __forceinline__ float g(float r, int k) const {
    const float diff = r - (float)k * delta;
    float v;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(v) : "f"(neg_gamma_l2e * diff * diff));
    return v;
  }
  // u' g_k + u g_k' = g_k (u' - 2 gamma u (r - k Delta))
  __device__ __forceinline__ float dug(float r, int k, float u, float du) const {
    const float diff = r - (float)k * delta;
    return g(r, k) * fmaf(-two_gamma * u, diff, du);
  }
};
// 8 consecutive floats (one 32-byte sector) per lane in ONE request: the rows of a gather are 512 bytes apart, so every lane
// costs an L1 tag cycle per instruction, and a 256-bit access halves the instructions
__device__ __forceinline__ void ldg8(const float* p, float* v) {
  asm volatile("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
               : "l"(p));
}
__device__ __forceinline__ void stg8(float* p, const float* v) {
  asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "r"(__float_as_uint(v[0])),
               "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])),
               "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7]))
               : "memory");
}
template <int N>
__device__ __forceinline__ void ldgN(const float* p, float (&v)[N]) {
  if constexpr (N == 8) ldg8(p, v);
  else {
    const float4 x = __ldg(reinterpret_cast<const float4*>(p));
    v[0] = x.x; v[1] = x.y; v[2] = x.z; v[3] = x.w;
  }
}
template <int N>
__device__ __forceinline__ void stgN(float* p, const float (&v)[N]) {
  if constexpr (N == 8) stg8(p, v);
  else *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}

// the six product terms of one K = 16 step: a1 b1 into the main accumulator, the five small ones (smallest first) into the other
template <class FA, class FB>
__device__ __forceinline__ void mma6(uint32_t d_main, uint32_t d_small, FA a_desc, FB b_desc, uint32_t idesc, bool accumulate) {
  constexpr int IA[5] = {2, 1, 0, 1, 0}, IB[5] = {0, 1, 2, 0, 1};
#pragma unroll
  for (int t = 0; t < 5; ++t) tc::mma_bf16(d_small, a_desc(IA[t]), b_desc(IB[t]), idesc, accumulate || t > 0);
  tc::mma_bf16(d_main, a_desc(0), b_desc(0), idesc, accumulate);
}

// Shared-memory fallback of the segmented sum (more than MAX_SEG receivers in the tile): thread = channel
__device__ __forceinline__ void segmented_store_x3(const unsigned char* A, const int* __restrict__ recv_s,
                                                   const int32_t* __restrict__ rowptr, int64_t e0, int64_t tile,
                                                   float* __restrict__ out, float* __restrict__ head, float* __restrict__ tail,
                                                   int c) {
  int cur = recv_s[0];
  float sum = 0.f;
  const uint32_t coff = (uint32_t)((c >> 6) * SLAB + (c & 7) * 2);
  const int cc = (c & 63) >> 3;
  for (int e = 0; e <= TE; ++e) {
    const int rcv = e < TE ? recv_s[e] : -2;
    if (rcv != cur) {
      if (cur >= 0) {
        const int64_t s0 = rowptr[cur], s1 = rowptr[cur + 1];
        if (s0 >= e0 && s1 <= e0 + TE) out[(size_t)cur * D + c] = sum;
        else if (s0 < e0) head[(size_t)tile * D + c] = sum;
        else tail[(size_t)tile * D + c] = sum;
      }
      cur = rcv;
      sum = 0.f;
    }
    if (e < TE && rcv >= 0) {
      const uint32_t o = coff + e * 128 + ((cc ^ (e & 7)) << 4);
      float v = 0.f;
#pragma unroll
      for (int i = 2; i >= 0; --i) v += __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(A + i * (NCH * SLAB) + o));
      sum += v;
    }
  }
}

template <bool BWD>
__global__ void __launch_bounds__(NT, 1) k_edge_x3(EdgeArgs a, int64_t n_tiles_cap, const __nv_bfloat16* __restrict__ W2x3,
                                                   const __nv_bfloat16* __restrict__ W13x3) {
  extern __shared__ unsigned char smem_raw[];
  const int64_t n_edges = a.E_dyn ? (int64_t)__ldg(a.E_dyn) : a.E;
  const int64_t n_tiles = a.E_dyn ? (n_edges + TE - 1) / TE : n_tiles_cap;
  const uint32_t base = (tc::smem_u32(smem_raw) + 1023u) & ~1023u;
  unsigned char* gen = smem_raw + (base - tc::smem_u32(smem_raw));
  int* recv_s = reinterpret_cast<int*>(gen + SM::recv);
  float* w_s = reinterpret_cast<float*>(gen + SM::w);
  float* ubar_s = reinterpret_cast<float*>(gen + SM::ubar);
  Seg& G = *reinterpret_cast<Seg*>(gen + SM::seg);
  uint32_t* slot = reinterpret_cast<uint32_t*>(gen + SM::slot);
  unsigned char* Aop = gen + SM::A;
  auto bar = [&](int i) -> uint32_t { return base + SM::bar + 8u * (uint32_t)i; };

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  // ---- one-time setup: resident weight images, barriers, TMEM ----
  {
    const uint4* src = reinterpret_cast<const uint4*>(W2x3);
    uint4* dst = reinterpret_cast<uint4*>(gen + SM::w2);
    for (int i = tid; i < 3 * D * D * 2 / 16; i += NT) dst[i] = __ldg(src + i);
    src = reinterpret_cast<const uint4*>(W13x3);
    dst = reinterpret_cast<uint4*>(gen + SM::w13);
    for (int i = tid; i < 3 * D * K1 * 2 / 16; i += NT) dst[i] = __ldg(src + i);
  }
  if (tid == 0) {
    tc::mbar_init(bar(B_A0), N_EPI_WARPS);
    for (int s = 0; s < 4 * NCH; ++s) tc::mbar_init(bar(B_S + s), CPS == 8 ? 8 : 16);
    tc::mbar_init(bar(B_G1), 1); tc::mbar_init(bar(B_G2), 1); tc::mbar_init(bar(B_G3), 1); tc::mbar_init(bar(B_FIN), 1);
    tc::mbar_init(bar(B_SEG), 1); tc::mbar_init(bar(B_RO), N_EPI_WARPS);
    tc::fence_mbar_init();
  }
  if (warp == 0) tc::tmem_alloc<TMEM_COLS>(slot);
  tc::fence_proxy_async();
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *slot;
  const uint32_t TX = tmem, TXs = tmem + D, TY = tmem + 2 * D, TYs = tmem + 3 * D;
  const uint32_t TS = TY, TSs = TY + 16, T4 = TY + 32, T4s = TY + 64;   // GS and G4 outputs over the dead head of Y

  if (blockIdx.x >= n_tiles) {
    // no tile for this CTA (only possible with E_dyn: the grid is sized from the capacity)
  } else if (warp == MMA_WARP) {
    // ====== MMA issuer: the whole warp follows the barriers, one elected lane issues ======
    constexpr uint32_t IDESC_ND = tc::idesc_bf16(128, D, 0, 0);
    constexpr uint32_t IDESC_ND_BT = tc::idesc_bf16(128, D, 0, 1);
    constexpr uint32_t IDESC_N32_BT = tc::idesc_bf16(128, K1, 0, 1);
    constexpr uint32_t IDESC_SEG = tc::idesc_bf16(128, 16, 1, 0);
    uint32_t ph_a0 = 0, ph_seg = 0, ph_ro = 0, ph_s = 0;  // parities of the next completion of B_A0 / B_SEG / B_S + i (bit i)
    auto wait_kstep = [&](int s, int kk) {
      tc::mbar_wait(bar(B_S + 4 * s + kk), (ph_s >> (4 * s + kk)) & 1u);
      ph_s ^= 1u << (4 * s + kk);
      tc::fence_after_sync();
    };
    auto a_slab = [&](int i, int s, int kk) {
      return tc::smem_desc(base + SM::A + i * (NCH * SLAB) + s * SLAB + kk * 32, 16, 1024, tc::LAYOUT_SW128);
    };
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      // A0 of this tile written by every epilogue warp; G4 / GS of the previous tile are complete (the epilogue waited
      // for B_FIN before it overwrote the slabs), so X is free
      tc::mbar_wait(bar(B_A0), ph_a0);
      ph_a0 ^= 1u;
      tc::fence_after_sync();
      if (tc::elect_one()) {
#pragma unroll
        for (int kk = 0; kk < K1 / 16; ++kk)
          mma6(TX, TXs, [&](int i) { return tc::smem_desc(base + SM::A + i * (TE * K1 * 2) + kk * 256, 128, 512, tc::LAYOUT_NONE); },
               [&](int i) { return tc::smem_desc(base + SM::w13 + i * (D * K1 * 2) + kk * 256, 128, 512, tc::LAYOUT_NONE); },
               IDESC_ND, kk != 0);
        tc::mma_commit(bar(B_G1));
      }
      __syncwarp();
      // ---- G2: Y = s . W2^T, one K step (16 channels) at a time. Its accumulators hold the outputs of GS / G4 of the
      // previous tile until every epilogue warp has read them out ----
      if (tile != blockIdx.x) {
        tc::mbar_wait(bar(B_RO), ph_ro);
        ph_ro ^= 1u;
      }
#pragma unroll
      for (int s = 0; s < NCH; ++s) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          wait_kstep(s, kk);
          if (tc::elect_one()) {
            mma6(TY, TYs, [&](int i) { return a_slab(i, s, kk); },
                 [&](int i) { return tc::smem_desc(base + SM::w2 + i * (D * D * 2) + s * (D * 128) + kk * 32, 16, 1024, tc::LAYOUT_SW128); },
                 IDESC_ND, (s | kk) != 0);
            if (s == NCH - 1 && kk == 3) tc::mma_commit(bar(B_G2));
          }
          __syncwarp();
        }
      }
      if (BWD) {
        // ---- G3: X = pbar . W2 (the W2 images read MN-major) ----
#pragma unroll
        for (int s = 0; s < NCH; ++s) {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) {
            wait_kstep(s, kk);
            if (tc::elect_one()) {
              mma6(TX, TXs, [&](int i) { return a_slab(i, s, kk); },
                   [&](int i) { return tc::smem_desc(base + SM::w2 + i * (D * D * 2) + (4 * s + kk) * 2048, D * 128, 1024, tc::LAYOUT_SW128); },
                   IDESC_ND_BT, (s | kk) != 0);
              if (s == NCH - 1 && kk == 3) tc::mma_commit(bar(B_G3));
            }
            __syncwarp();
          }
        }
      }
      // ---- G4 (reverse): [ebar | tbar] = abar . [W1c | W3]; B = the G1 images [channel][32] read MN-major (N = 32,
      // K = channel): K-direction 8-channel group stride (LBO) 512 B, N-direction core-matrix stride (SBO) 128 B ----
#pragma unroll
      for (int s = 0; s < NCH; ++s) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          wait_kstep(s, kk);
          if (BWD && tc::elect_one()) {
            mma6(T4, T4s, [&](int i) { return a_slab(i, s, kk); },
                 [&](int i) { return tc::smem_desc(base + SM::w13 + i * (D * K1 * 2) + (4 * s + kk) * 1024, 512, 128, tc::LAYOUT_NONE); },
                 IDESC_N32_BT, (s | kk) != 0);
          }
          __syncwarp();
        }
      }
      // ---- GS: segmented sum of the slabs (phi / abar) with the 0/1 selector of the segment warp ----
      tc::mbar_wait(bar(B_SEG), ph_seg);
      ph_seg ^= 1u;
      tc::fence_after_sync();
      const int R = *reinterpret_cast<volatile int*>(&G.R);
      if (tc::elect_one()) {
        if (R <= MAX_SEG) {
#pragma unroll
          for (int j = 0; j < TE / 16; ++j) {
            const uint64_t sel_d = tc::smem_desc(base + SM::sel + j * 256, 128, 2048, tc::LAYOUT_NONE);
#pragma unroll
            for (int t = 2; t >= 0; --t)
              tc::mma_bf16(t == 0 ? TS : TSs, tc::smem_desc(base + SM::A + t * (NCH * SLAB) + j * 2048, SLAB, 1024, tc::LAYOUT_SW128),
                           sel_d, IDESC_SEG, t == 0 ? j != 0 : (j != 0 || t != 2));
          }
        }
        tc::mma_commit(bar(B_FIN));
      }
      __syncwarp();
    }
  } else if (warp == SEG_WARP) {
    // ====== segment analysis: receivers of the tile in order of appearance, destination of each sum, 0/1 selector ======
    uint32_t ph_ro = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      const int64_t e0 = tile * TE;
      int rcv[4], prv[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int64_t ge = e0 + lane + 32 * k;
        rcv[k] = ge < n_edges ? __ldg(a.recv + ge) : -1;
        prv[k] = (ge < n_edges && ge > e0) ? __ldg(a.recv + ge - 1) : -2;
      }
      uint32_t fm[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) fm[k] = __ballot_sync(0xffffffffu, rcv[k] >= 0 && rcv[k] != prv[k]);
      int rloc[4];
      int64_t s0[4], s1[4];
      int before = 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        rloc[k] = before + __popc(fm[k] & (0xffffffffu >> (31 - lane))) - 1;
        const bool first = ((fm[k] >> lane) & 1u) && rloc[k] < MAX_SEG;
        s0[k] = first ? __ldg(a.rowptr + rcv[k]) : 0;
        s1[k] = first ? __ldg(a.rowptr + rcv[k] + 1) : -1;   // s1 < 0: not the first edge of a receiver
        before += __popc(fm[k]);
      }
      // the selector and the segment table are free once every epilogue warp has read out the previous tile
      if (tile != blockIdx.x) {
        tc::mbar_wait_warp(bar(B_RO), ph_ro);
        ph_ro ^= 1u;
      }
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (s1[k] >= 0)
          G.dst[rloc[k]] = (s0[k] >= e0 && s1[k] <= e0 + TE) ? (BWD ? a.Pbar : a.m) + (size_t)rcv[k] * D
                                                            : (s0[k] < e0 ? a.head : a.tail) + (size_t)tile * D;
      if (lane == 0) G.R = before;
      uint4* z = reinterpret_cast<uint4*>(gen + SM::sel);
#pragma unroll
      for (int i = 0; i < MAX_SEG * TE * 2 / 16 / 32; ++i) z[lane + 32 * i] = make_uint4(0u, 0u, 0u, 0u);
      __syncwarp();
      // Sel (r, e) -> (r/8)*2048 + (e/8)*128 + (r%8)*16 + (e%8)*2
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int e = lane + 32 * k;
        if (rcv[k] >= 0 && rloc[k] < MAX_SEG)
          *reinterpret_cast<unsigned short*>(gen + SM::sel + (rloc[k] >> 3) * 2048 + (e >> 3) * 128 + (rloc[k] & 7) * 16 +
                                             (e & 7) * 2) = (unsigned short)0x3F80;  // bf16 1.0
      }
      tc::fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_SEG));
    }
  } else {
    // =========================== epilogue warps ===========================
    const int q = warp & 3, g = warp >> 2;
    const int row = q * 32 + lane;
    const uint32_t tlane = (uint32_t)(q * 32) << 16;
    // step j of a phase: this thread's CPS channels ch(j) .. ch(j) + CPS - 1 of K step kst(j). CPS = 8: two K steps in
    // progress at a time (8 warps each); CPS = 4: one (all 16 warps), the tensor core trails by a single K step
    constexpr int NSTEP = D / (4 * CPS);
    auto kst = [&](int j) { return CPS == 8 ? 2 * j + (g >> 1) : j; };
    auto ch = [&](int j) { return CPS == 8 ? 16 * kst(j) + 8 * (g & 1) : 16 * j + 4 * g; };
    auto soff = [&](int j) {  // byte offset of those 2 CPS bytes inside an operand term (SW128 slabs of 64 channels)
      const int k = kst(j);
      const int chunk = (k & 3) * 2 + (CPS == 8 ? (g & 1) : (g >> 1));
      return (uint32_t)((k >> 2) * SLAB + row * 128 + ((chunk ^ (row & 7)) << 4) + (CPS == 8 ? 0 : 8 * (g & 1)));
    };
    const Rbf rbf(a.r_cut, a.n_rbf);
    uint32_t ph = 0;  // bit i: parity of the next completion of barrier i
    auto wait_bar = [&](int i) {
      tc::mbar_wait_warp(bar(i), (ph >> i) & 1u);
      ph ^= 1u << i;
      tc::fence_after_sync();
    };
    // this warp's part of an operand is written (shared memory -> async proxy) and its tensor-memory reads are done
    auto publish = [&](int i) {
      tc::fence_proxy_async();
      tc::fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(i));
    };
    // row metadata of a tile: fetched one tile ahead by every thread of the row
    int rc_n = -1, sd_n = 0;
    float r_n = 0.f;
    auto fetch_meta = [&](int64_t tile) {
      const int64_t e = tile * TE + row;
      rc_n = -1; sd_n = 0; r_n = 0.f;
      if (tile < n_tiles && e < n_edges) { rc_n = __ldg(a.recv + e); sd_n = __ldg(a.send + e); r_n = __ldg(&a.rvec[e].w); }
    };
    // P0 of a tile: features computed in registers (under the last MMAs of the previous tile), stored once the operand
    // region is free. A0 (row, k) -> (row/8)*512 + (k/8)*128 + (row%8)*16 + (k%8)*2, split i at i * 8192; column group g
    // writes k = 8g..8g+7
    struct Feat { uint32_t p[3][4]; float u, du; };
    auto features = [&](int64_t tile, int rc, float r_e, Feat& o) {
      float f[8];
      o.u = 0.f; o.du = 0.f;
      if (g < 2) {
        if (rc >= 0) envelope_f(r_e, a.r_cut, o.u, o.du);
#pragma unroll
        for (int k = 0; k < 8; ++k) f[k] = 8 * g + k < a.n_rbf ? o.u * rbf.g(r_e, 8 * g + k) : 0.f;   // u = 0 beyond the edge list
      } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) f[k] = 0.f;
        if (a.t3 && rc >= 0) ldg8(a.t3 + (size_t)(tile * TE + row) * 16 + 8 * (g - 2), f);
      }
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        uint32_t h[3];
        split3(f[2 * t], f[2 * t + 1], h);
        o.p[0][t] = h[0]; o.p[1][t] = h[1]; o.p[2][t] = h[2];
      }
    };
    auto store_a0 = [&](const Feat& o, int rc) {
      if (g == 0) { recv_s[row] = rc; w_s[row] = a.alpha * o.u; }
#pragma unroll
      for (int i = 0; i < 3; ++i)
        *reinterpret_cast<uint4*>(Aop + i * (TE * K1 * 2) + (row >> 3) * 512 + g * 128 + (row & 7) * 16) =
            make_uint4(o.p[i][0], o.p[i][1], o.p[i][2], o.p[i][3]);
      publish(B_A0);
    };
    // Read-out of a finished tile (segment sums out of Yseg, E4), deferred until A0 of the NEXT tile is published so that
    // it runs under that tile's G1 instead of ending every tile with idle tensor cores.
    auto read_out = [&](int64_t tile, bool valid, float r_e, float u, float du) {
      const int64_t e0 = tile * TE;
      const int R = G.R;
      if (R <= MAX_SEG && g == 0) {
        float acc[16];
        tmem_ld_sum<16>(TS + tlane, TSs + tlane, acc);
#pragma unroll
        for (int r = 0; r < MAX_SEG; ++r)
          if (r < R) G.dst[r][row] = acc[r];
      }
      if (BWD && g == 1) {
        // E4; one addition per edge and launch: a fire-and-forget reduction is deterministic and has no load latency
        float eb[16];
        tmem_ld_sum<16>(T4 + tlane, T4s + tlane, eb);
        if (valid) {
          float part = 0.f;
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            if (k < a.n_rbf) part = fmaf(eb[k], rbf.dug(r_e, k, u, du), part);
          }
          const float ubar = a.alpha * ((ubar_s[row] + ubar_s[TE + row]) + (ubar_s[2 * TE + row] + ubar_s[3 * TE + row]));
          atomicAdd(a.rbar + e0 + row, fmaf(ubar, du, part));
        }
      }
      if (BWD && g == 2 && a.tbar) {
        float tb[16];
        tmem_ld_sum<16>(T4 + tlane + 16u, T4s + tlane + 16u, tb);
        if (valid) {
          stg8(a.tbar + (size_t)(e0 + row) * 16, tb);
          stg8(a.tbar + (size_t)(e0 + row) * 16 + 8, tb + 8);
        }
      }
      // the segment table, Yseg, D4 and the u-bar partials of the tile are read: the segment warp, the next GS / G4 and
      // the next E2 may overwrite them
      tc::fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_RO));
    };

    fetch_meta(blockIdx.x);
    float u_e, du_e;
    {
      Feat ft;
      features(blockIdx.x, rc_n, r_n, ft);
      store_a0(ft, rc_n);
      u_e = ft.u; du_e = ft.du;
    }
    bool ro_valid = false;
    float ro_r = 0.f, ro_u = 0.f, ro_du = 0.f;

    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      const int64_t e0 = tile * TE;
      const int rc = rc_n, sd = sd_n;
      const float r_e = r_n;
      const bool valid = rc >= 0;
      // sender rows Q_j: random rows out of L2; the first step is requested before anything else of the tile is computed
      const float* Qrow = a.Q + (size_t)sd * a.ldq;
      const float* Prow = a.P + (size_t)(valid ? rc : 0) * a.ldp;
      float qf[CPS], pf[CPS];
      ldgN<CPS>(Qrow + ch(0), qf);
      ldgN<CPS>(Prow + ch(0), pf);
      fetch_meta(tile + gridDim.x);
      if (tile != blockIdx.x) read_out(tile - gridDim.x, ro_valid, ro_r, ro_u, ro_du);
      ro_valid = valid; ro_r = r_e; ro_u = u_e; ro_du = du_e;
      // ================= E1 =================
      float ds[BWD ? NSTEP : 1][CPS];
      wait_bar(B_G1);
#pragma unroll
      for (int j = 0; j < NSTEP; ++j) {
        float v[CPS];
        tmem_ld_sum<CPS>(TX + tlane + (uint32_t)ch(j), TXs + tlane + (uint32_t)ch(j), v);
#pragma unroll
        for (int k = 0; k < CPS; ++k) v[k] += pf[k] + qf[k];
        if (j + 1 < NSTEP) { ldgN<CPS>(Prow + ch(j + 1), pf); ldgN<CPS>(Qrow + ch(j + 1), qf); }
#pragma unroll
        for (int k = 0; k < CPS; ++k) {
          if (BWD) silu_both_x3(v[k], v[k], ds[j][k]);
          else v[k] = silu_x3(v[k]);
        }
        store_split<CPS>(Aop, soff(j), v);
        publish(B_S + kst(j));
      }
      // ================= E2 =================
      wait_bar(B_G2);
      if (!BWD) {
        const float wr = w_s[row];
#pragma unroll
        for (int j = 0; j < NSTEP; ++j) {
          float y[CPS];
          tmem_ld_sum<CPS>(TY + tlane + (uint32_t)ch(j), TYs + tlane + (uint32_t)ch(j), y);
          float bb[CPS];   // b2 lives in the weight blob: 16-byte aligned only, no 256-bit load
#pragma unroll
          for (int k4 = 0; k4 < CPS / 4; ++k4) {
            const float4 b = __ldg(reinterpret_cast<const float4*>(a.b2 + ch(j)) + k4);
            bb[4 * k4] = b.x; bb[4 * k4 + 1] = b.y; bb[4 * k4 + 2] = b.z; bb[4 * k4 + 3] = b.w;
          }
#pragma unroll
          for (int k = 0; k < CPS; ++k) y[k] = wr * silu_x3(y[k] + bb[k]);
          store_split<CPS>(Aop, soff(j), y);
          publish(B_S + kst(j));
        }
      } else {
        const float au = w_s[row];
        const float* Mrow = a.mbar + (size_t)(valid ? rc : 0) * D;
        float up = 0.f;
        float mb[CPS];
        ldgN<CPS>(Mrow + ch(0), mb);
#pragma unroll
        for (int j = 0; j < NSTEP; ++j) {
          float y[CPS];
          tmem_ld_sum<CPS>(TY + tlane + (uint32_t)ch(j), TYs + tlane + (uint32_t)ch(j), y);
          float bb[CPS];   // b2 lives in the weight blob: 16-byte aligned only, no 256-bit load
#pragma unroll
          for (int k4 = 0; k4 < CPS / 4; ++k4) {
            const float4 b = __ldg(reinterpret_cast<const float4*>(a.b2 + ch(j)) + k4);
            bb[4 * k4] = b.x; bb[4 * k4 + 1] = b.y; bb[4 * k4 + 2] = b.z; bb[4 * k4 + 3] = b.w;
          }
#pragma unroll
          for (int k = 0; k < CPS; ++k) {
            float phi, dphi;
            silu_both_x3(y[k] + bb[k], phi, dphi);
            up = fmaf(mb[k], phi, up);
            y[k] = au * mb[k] * dphi;
          }
          if (j + 1 < NSTEP) ldgN<CPS>(Mrow + ch(j + 1), mb);
          store_split<CPS>(Aop, soff(j), y);
          if (j == NSTEP - 1) ubar_s[g * TE + row] = up;
          publish(B_S + kst(j));
        }
        // ================= E3 =================
        wait_bar(B_G3);
#pragma unroll
        for (int j = 0; j < NSTEP; ++j) {
          float x[CPS];
          tmem_ld_sum<CPS>(TX + tlane + (uint32_t)ch(j), TXs + tlane + (uint32_t)ch(j), x);
#pragma unroll
          for (int k = 0; k < CPS; ++k) ds[j][k] *= x[k];   // abar, kept for the spill below
          store_split<CPS>(Aop, soff(j), ds[j]);
          publish(B_S + kst(j));
        }
        // The fp32 spill goes out after the last step is published: the fences of publish() wait for global stores issued
        // before them (measured: 3.4 k cycles per slab). It drains under the wait for G4 / GS.
        if (valid) {
          float* dst = a.abar + (size_t)(e0 + row) * D;
#pragma unroll
          for (int j = 0; j < NSTEP; ++j) stgN<CPS>(dst + ch(j), ds[j]);
        }
      }
      // ================= P0 of the next tile under G4 / GS of this one =================
      const int64_t next = tile + gridDim.x;
      Feat ft;
      if (next < n_tiles) features(next, rc_n, r_n, ft);
      wait_bar(B_FIN);
      wait_bar(B_SEG);
      if (G.R > MAX_SEG) {  // rare: more receivers than the selector holds, sum the slabs before they are overwritten
        if (warp < D / 32)
          segmented_store_x3(Aop, recv_s, a.rowptr, e0, tile, BWD ? a.Pbar : a.m, a.head, a.tail, warp * 32 + lane);
        named_bar_sync(1, N_EPI_WARPS * 32);
      }
      if (next < n_tiles) { store_a0(ft, rc_n); u_e = ft.u; du_e = ft.du; }
    }
    read_out(n_tiles - 1 - (n_tiles - 1 - blockIdx.x) % gridDim.x, ro_valid, ro_r, ro_u, ro_du);
  }
  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<TMEM_COLS>(tmem);
}

// out[i] = tail[t] + head[t+1] + ... for the segment that starts in tile t and continues beyond it
__global__ void k_segment_fixup_x3(int64_t E, const int32_t* __restrict__ E_dyn, const int32_t* __restrict__ rowptr,
                                   const int32_t* __restrict__ recv, const float* __restrict__ head,
                                   const float* __restrict__ tail, float* __restrict__ out) {
  if (E_dyn) E = *E_dyn;
  const int64_t t = blockIdx.x;
  const int64_t e0 = t * TE, e1 = e0 + TE;
  if (e1 >= E) return;
  const int i = recv[e1 - 1];
  const int64_t s0 = rowptr[i], s1 = rowptr[i + 1];
  if (!(s1 > e1 && s0 >= e0)) return;
  const int c = threadIdx.x;
  float sum = tail[(size_t)t * D + c];
  for (int64_t t2 = t + 1; t2 * TE < s1; ++t2) sum += head[(size_t)t2 * D + c];
  out[(size_t)i * D + c] = sum;
}
}  // namespace

namespace {
template <bool BWD>
int launch_x3(mlip_ctx* ctx, const EdgeArgs& a) {
  const int64_t tiles = (a.E + TE - 1) / TE;
  if (tiles == 0) return MLIP_OK;
  const size_t smem = SM::bytes + 1024;  // + alignment slack
  const unsigned grid = (unsigned)(tiles < ctx->num_sms ? tiles : ctx->num_sms);
  MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_edge_x3<BWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_edge_x3<BWD><<<grid, NT, smem, ctx->stream>>>(a, tiles, a.W2x3, a.W13x3);
  k_segment_fixup_x3<<<(unsigned)tiles, D, 0, ctx->stream>>>(a.E, a.E_dyn, a.rowptr, a.recv, a.head, a.tail, BWD ? a.Pbar : a.m);
  ctx->launches += 2;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
}  // namespace

bool mlip_edge_x3_supported(int d, const EdgeArgs& a) { return d == D && a.W2x3 && a.W13x3; }
int mlip_edge_forward_x3(mlip_ctx* ctx, const EdgeArgs& a) { return launch_x3<false>(ctx, a); }
int mlip_edge_backward_x3(mlip_ctx* ctx, const EdgeArgs& a) { return launch_x3<true>(ctx, a); }
