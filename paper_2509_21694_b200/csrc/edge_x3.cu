// MLIP_FP32 path of the fused edge kernels (A6, A7, edge part of A10) on the tensor cores, d = 128: every
// contraction runs on tcgen05 with fp32 operands SPLIT INTO THREE bf16 TERMS, x = x1 + x2 + x3 with
// x1 = bf16(x), x2 = bf16(x - x1), x3 = bf16(x - x1 - x2) (24 significant bits, the exponent range of fp32: no
// range contract as in the MLIP_BF16 path). A product a b is evaluated as the six terms a1 b1 + a1 b2 + a2 b1 +
// a1 b3 + a2 b2 + a3 b1 accumulated in fp32 in tensor memory; what is dropped is below 2^-24 |a b|. Six bf16 MMAs
// at 8192 flop/clk/SM replace fp32 FMAs at 256 flop/clk/SM. Everything between the contractions (gathers, SiLU,
// envelope, radial basis) is the fp32 arithmetic of edge_f32.cu, so the two kernels agree to fp32 rounding.
//
// One persistent CTA per SM (16 warps, all in lock step, thread 0 issues the MMAs) walks over tiles of 128
// receiver-sorted edges. The split images of W2 [d,d] and of [W1c | W3] [d,32] stay in shared memory.
//   P0  edge metadata, envelope, radial basis; A0 = [e_hat | t_e] [128,32] split into three operand tiles;
//       receivers of the tile and the 0/1 selector of the segmented sum
//   G1  X = A0 . [W1c | W3]^T                               (K = 32; t_e = 0 without the three-body term)
//   E1  a = X + P_i + Q_j ; s = SiLU(a) -> split slabs ; the reverse pass keeps SiLU'(a) in registers
//   G2  Y = s . W2^T            issued per 64-channel K slab as soon as E1 has written it
//   E2  forward : phi = alpha u_e SiLU(Y + b2) -> split slabs
//       reverse : pbar = alpha u_e mbar_i SiLU'(p) -> split slabs ; ubar_e = alpha <mbar_i, phi_e>
//   G3  X = pbar . W2           (reverse; the same W2 images read MN-major)
//   E3  abar = X SiLU'(a) -> global spill (fp32, read back through rev[] by k_gather_rev_f32) and split slabs
//   G4  [ebar | tbar] = abar . [W1c | W3]   (N = 32, the G1 images read MN-major)
//   GS  segmented sum over runs of equal receiver as an MMA with the 0/1 selector (three terms: the selector is
//       exact): Yseg[channel, r] = slab^T . Sel ; m_i (forward) / Pbar_i (reverse). Tiles with more than 16
//       receivers sum the slabs in a shared-memory loop.
//   E4  rbar_e += ubar_e u' + sum_k ebar_k (u' g_k + u g'_k) ; tbar_e -> global
// Segments that straddle tiles go through per-tile head / tail rows and a fix-up kernel, as in edge_f32.cu. No
// floating-point atomics: results are bitwise reproducible.
#include <cuda_bf16.h>
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"
#include "tc_images.cuh"
#include "tc_ptx.cuh"

namespace {
constexpr int D = 128;            // channels (the only width this kernel is built for)
constexpr int TE = 128;           // edges per tile = MMA M
constexpr int NT = 512;           // threads: warp = (lane quarter q = warp % 4, column group g = warp / 4)
constexpr int NCH = D / 64;       // 64-channel operand slabs
constexpr int K1 = 32;            // K of G1: 16 radial + 16 angle terms
constexpr int SLAB = TE * 128;    // one [128 x 64] bf16 SW128 slab
constexpr int MAX_SEG = 16;       // receivers per tile handled by the selector MMA
constexpr int SEG_WARP = 15;

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
  static constexpr uint32_t recv = sel + MAX_SEG * TE * 2;        // int[128]
  static constexpr uint32_t send = recv + TE * 4;                 // int[128]
  static constexpr uint32_t u = send + TE * 4;                    // float[128] each: u, du, r, w = alpha u
  static constexpr uint32_t du = u + TE * 4;
  static constexpr uint32_t r = du + TE * 4;
  static constexpr uint32_t w = r + TE * 4;
  static constexpr uint32_t ubar = w + TE * 4;                    // float[4][128]
  static constexpr uint32_t seg = ubar + 4 * TE * 4;              // Seg
  static constexpr uint32_t bar = seg + sizeof(Seg);              // one mbarrier
  static constexpr uint32_t slot = bar + 8;                       // TMEM base address
  static constexpr uint32_t bytes = slot + 8;
  static_assert(bytes <= 232448, "shared memory budget of one SM exceeded");
};
constexpr int TMEM_COLS = 512;    // X [0,128) | Y [128,256) | Yseg [256,272) | D4 [288,320)

// x = h[0] + h[1] + h[2] (bf16 each), two values per register
__device__ __forceinline__ void split3(float x0, float x1, uint32_t (&h)[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    h[i] = tc::pack_bf16(x0, x1);
    if (i < 2) { x0 -= tc::bf16_lo(h[i]); x1 -= tc::bf16_hi(h[i]); }
  }
}
// 16 consecutive channels of one row -> the two 16-byte chunks of the three split slabs
__device__ __forceinline__ void store_split16(unsigned char* slab0, uint32_t so0, uint32_t so1, const float (&v)[16]) {
  uint32_t p[3][8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    uint32_t h[3];
    split3(v[2 * j], v[2 * j + 1], h);
    p[0][j] = h[0]; p[1][j] = h[1]; p[2][j] = h[2];
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    unsigned char* s = slab0 + i * (NCH * SLAB);
    *reinterpret_cast<uint4*>(s + so0) = make_uint4(p[i][0], p[i][1], p[i][2], p[i][3]);
    *reinterpret_cast<uint4*>(s + so1) = make_uint4(p[i][4], p[i][5], p[i][6], p[i][7]);
  }
}
__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// the six product terms of one K = 16 step, smallest first
template <class FA, class FB>
__device__ __forceinline__ void mma6(uint32_t d_tmem, FA a_desc, FB b_desc, uint32_t idesc, bool accumulate) {
  constexpr int IA[6] = {2, 1, 0, 1, 0, 0}, IB[6] = {0, 1, 2, 0, 1, 0};
#pragma unroll
  for (int t = 0; t < 6; ++t) tc::mma_bf16(d_tmem, a_desc(IA[t]), b_desc(IB[t]), idesc, accumulate || t > 0);
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
  int* send_s = reinterpret_cast<int*>(gen + SM::send);
  float* u_s = reinterpret_cast<float*>(gen + SM::u);
  float* du_s = reinterpret_cast<float*>(gen + SM::du);
  float* r_s = reinterpret_cast<float*>(gen + SM::r);
  float* w_s = reinterpret_cast<float*>(gen + SM::w);
  float* ubar_s = reinterpret_cast<float*>(gen + SM::ubar);
  Seg& G = *reinterpret_cast<Seg*>(gen + SM::seg);
  uint32_t* slot = reinterpret_cast<uint32_t*>(gen + SM::slot);
  unsigned char* Aop = gen + SM::A;
  const uint32_t bar = base + SM::bar;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int q = warp & 3, g = warp >> 2;
  const int row = q * 32 + lane;
  const uint32_t tlane = (uint32_t)(q * 32) << 16;
  const uint32_t so0 = (uint32_t)(row * 128 + (((2 * g) ^ (row & 7)) << 4));
  const uint32_t so1 = (uint32_t)(row * 128 + (((2 * g + 1) ^ (row & 7)) << 4));

  // ---- one-time setup: resident weight images, barrier, TMEM ----
  {
    const uint4* src = reinterpret_cast<const uint4*>(W2x3);
    uint4* dst = reinterpret_cast<uint4*>(gen + SM::w2);
    for (int i = tid; i < 3 * D * D * 2 / 16; i += NT) dst[i] = __ldg(src + i);
    src = reinterpret_cast<const uint4*>(W13x3);
    dst = reinterpret_cast<uint4*>(gen + SM::w13);
    for (int i = tid; i < 3 * D * K1 * 2 / 16; i += NT) dst[i] = __ldg(src + i);
  }
  if (tid == 0) { tc::mbar_init(bar, 1); tc::fence_mbar_init(); }
  if (warp == 0) tc::tmem_alloc<TMEM_COLS>(slot);
  tc::fence_proxy_async();
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *slot;
  const uint32_t TX = tmem, TY = tmem + D, TS = tmem + 2 * D, T4 = tmem + 2 * D + 32;
  uint32_t phase = 0;
  // all MMAs issued so far are complete and their results visible to every thread
  auto mma_done = [&]() {
    if (tid == 0) tc::mma_commit(bar);
    tc::mbar_wait_warp(bar, phase);
    phase ^= 1u;
    tc::fence_after_sync();
  };
  // shared-memory operands written by all threads -> visible to the tensor core; tensor-memory reads of all threads done
  auto operands_ready = [&]() {
    tc::fence_proxy_async();
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
  };
  constexpr uint32_t IDESC_ND = tc::idesc_bf16(128, D, 0, 0);
  constexpr uint32_t IDESC_ND_BT = tc::idesc_bf16(128, D, 0, 1);
  constexpr uint32_t IDESC_N32_BT = tc::idesc_bf16(128, K1, 0, 1);
  constexpr uint32_t IDESC_SEG = tc::idesc_bf16(128, 16, 1, 0);
  const float4* b2v = reinterpret_cast<const float4*>(a.b2);

  // row metadata of a tile: fetched one tile ahead by every thread of the row
  int rc_n = -1, sd_n = 0;
  float r_n = 0.f;
  auto fetch_meta = [&](int64_t tile) {
    const int64_t e = tile * TE + row;
    rc_n = -1; sd_n = 0; r_n = 0.f;
    if (tile < n_tiles && e < n_edges) { rc_n = __ldg(a.recv + e); sd_n = __ldg(a.send + e); r_n = __ldg(&a.rvec[e].w); }
  };
  fetch_meta(blockIdx.x);

  for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int64_t e0 = tile * TE;
    const int rc = rc_n, sd = sd_n;
    const float r_e = r_n;
    const bool valid = rc >= 0;
    // sender rows Q_j: random rows out of L2, requested before anything else of the tile is computed
    float4 qf[NCH][4];
    {
      const float* Qrow = a.Q + (size_t)sd * a.ldq + 16 * g;
#pragma unroll
      for (int s = 0; s < NCH; ++s)
#pragma unroll
        for (int k4 = 0; k4 < 4; ++k4) qf[s][k4] = ldg4(Qrow + 64 * s + 4 * k4);
    }
    fetch_meta(tile + gridDim.x);
    // ================= P0: metadata, features, selector =================
    // A0 (row, k) -> (row/8)*512 + (k/8)*128 + (row%8)*16 + (k%8)*2, split i at i * 8192; column group g writes k = 8g..8g+7
    {
      float f[8];
      if (g < 2) {
        float u = 0.f, du = 0.f;
        if (valid) envelope_f(r_e, a.r_cut, u, du);
        if (g == 0) {
          recv_s[row] = rc; send_s[row] = sd; u_s[row] = u; du_s[row] = du; r_s[row] = r_e; w_s[row] = a.alpha * u;
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          float gk = 0.f, dg;
          if (valid && 8 * g + k < a.n_rbf) rbf_f(r_e, a.r_cut, a.n_rbf, 8 * g + k, gk, dg);
          f[k] = u * gk;
        }
      } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) f[k] = 0.f;
        if (a.t3 && valid) {
          const float4 v0 = ldg4(a.t3 + (size_t)(e0 + row) * 16 + 8 * (g - 2)), v1 = ldg4(a.t3 + (size_t)(e0 + row) * 16 + 8 * (g - 2) + 4);
          f[0] = v0.x; f[1] = v0.y; f[2] = v0.z; f[3] = v0.w; f[4] = v1.x; f[5] = v1.y; f[6] = v1.z; f[7] = v1.w;
        }
      }
      uint32_t p[3][4];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        uint32_t h[3];
        split3(f[2 * t], f[2 * t + 1], h);
        p[0][t] = h[0]; p[1][t] = h[1]; p[2][t] = h[2];
      }
#pragma unroll
      for (int i = 0; i < 3; ++i)
        *reinterpret_cast<uint4*>(Aop + i * (TE * K1 * 2) + (row >> 3) * 512 + g * 128 + (row & 7) * 16) =
            make_uint4(p[i][0], p[i][1], p[i][2], p[i][3]);
    }
    if (warp == SEG_WARP) {
      // receivers of the tile in order of appearance, destination of each segment sum, 0/1 selector
      int rcv[4];
      uint32_t fm[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int e = lane + 32 * k;
        const int64_t ge = e0 + e;
        bool flag = false;
        rcv[k] = -1;
        if (ge < n_edges) {
          rcv[k] = a.recv[ge];
          flag = e == 0 || a.recv[ge - 1] != rcv[k];
        }
        fm[k] = __ballot_sync(0xffffffffu, flag);
      }
      int rloc[4];
      int before = 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        rloc[k] = before + __popc(fm[k] & (0xffffffffu >> (31 - lane))) - 1;
        if (((fm[k] >> lane) & 1u) && rloc[k] < MAX_SEG) {
          const int64_t s0 = a.rowptr[rcv[k]], s1 = a.rowptr[rcv[k] + 1];
          G.dst[rloc[k]] = (s0 >= e0 && s1 <= e0 + TE) ? (BWD ? a.Pbar : a.m) + (size_t)rcv[k] * D
                                                       : (s0 < e0 ? a.head : a.tail) + (size_t)tile * D;
        }
        before += __popc(fm[k]);
      }
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
    }
    operands_ready();
    // ================= G1 =================
    if (tid == 0) {
#pragma unroll
      for (int kk = 0; kk < K1 / 16; ++kk)
        mma6(TX, [&](int i) { return tc::smem_desc(base + SM::A + i * (TE * K1 * 2) + kk * 256, 128, 512, tc::LAYOUT_NONE); },
             [&](int i) { return tc::smem_desc(base + SM::w13 + i * (D * K1 * 2) + kk * 256, 128, 512, tc::LAYOUT_NONE); },
             IDESC_ND, kk != 0);
    }
    mma_done();
    // ================= E1 / G2 =================
    float ds[BWD ? NCH : 1][16];
    {
      const float* Prow = a.P + (size_t)(valid ? rc : 0) * a.ldp + 16 * g;
#pragma unroll
      for (int s = 0; s < NCH; ++s) {
        float x[16];
        tc::tmem_ld16(TX + tlane + (uint32_t)(64 * s + 16 * g), x);
        float v[16];
#pragma unroll
        for (int k4 = 0; k4 < 4; ++k4) {
          const float4 p = ldg4(Prow + 64 * s + 4 * k4), qv = qf[s][k4];
          v[4 * k4] = p.x + qv.x + x[4 * k4]; v[4 * k4 + 1] = p.y + qv.y + x[4 * k4 + 1];
          v[4 * k4 + 2] = p.z + qv.z + x[4 * k4 + 2]; v[4 * k4 + 3] = p.w + qv.w + x[4 * k4 + 3];
        }
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          float sv, dv;
          silu_both_f(v[k], sv, dv);
          v[k] = valid ? sv : 0.f;
          if (BWD) ds[s][k] = valid ? dv : 0.f;
        }
        store_split16(Aop + s * SLAB, so0, so1, v);
        operands_ready();
        if (tid == 0) {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
            mma6(TY, [&](int i) { return tc::smem_desc(base + SM::A + i * (NCH * SLAB) + s * SLAB + kk * 32, 16, 1024, tc::LAYOUT_SW128); },
                 [&](int i) { return tc::smem_desc(base + SM::w2 + i * (D * D * 2) + s * (D * 128) + kk * 32, 16, 1024, tc::LAYOUT_SW128); },
                 IDESC_ND, (s | kk) != 0);
        }
      }
    }
    mma_done();
    // ================= E2 =================
    if (!BWD) {
      const float wr = w_s[row];
#pragma unroll
      for (int s = 0; s < NCH; ++s) {
        float y[16];
        tc::tmem_ld16(TY + tlane + (uint32_t)(64 * s + 16 * g), y);
#pragma unroll
        for (int k4 = 0; k4 < 4; ++k4) {
          const float4 b = __ldg(b2v + 16 * s + 4 * g + k4);
          y[4 * k4] = wr * silu_f(y[4 * k4] + b.x); y[4 * k4 + 1] = wr * silu_f(y[4 * k4 + 1] + b.y);
          y[4 * k4 + 2] = wr * silu_f(y[4 * k4 + 2] + b.z); y[4 * k4 + 3] = wr * silu_f(y[4 * k4 + 3] + b.w);
        }
        store_split16(Aop + s * SLAB, so0, so1, y);
      }
      operands_ready();
    } else {
      const float au = w_s[row];
      const float* Mrow = a.mbar + (size_t)(valid ? rc : 0) * D + 16 * g;
      float up = 0.f;
#pragma unroll
      for (int s = 0; s < NCH; ++s) {
        float y[16];
        tc::tmem_ld16(TY + tlane + (uint32_t)(64 * s + 16 * g), y);
#pragma unroll
        for (int k4 = 0; k4 < 4; ++k4) {
          const float4 b = __ldg(b2v + 16 * s + 4 * g + k4);
          float4 mb = ldg4(Mrow + 64 * s + 4 * k4);
          if (!valid) mb = make_float4(0.f, 0.f, 0.f, 0.f);
          float phi, dphi;
          silu_both_f(y[4 * k4] + b.x, phi, dphi); up = fmaf(mb.x, phi, up); y[4 * k4] = au * mb.x * dphi;
          silu_both_f(y[4 * k4 + 1] + b.y, phi, dphi); up = fmaf(mb.y, phi, up); y[4 * k4 + 1] = au * mb.y * dphi;
          silu_both_f(y[4 * k4 + 2] + b.z, phi, dphi); up = fmaf(mb.z, phi, up); y[4 * k4 + 2] = au * mb.z * dphi;
          silu_both_f(y[4 * k4 + 3] + b.w, phi, dphi); up = fmaf(mb.w, phi, up); y[4 * k4 + 3] = au * mb.w * dphi;
        }
        store_split16(Aop + s * SLAB, so0, so1, y);
        if (s == NCH - 1) ubar_s[g * TE + row] = up;
        operands_ready();
        // ================= G3: X = pbar . W2 (W2 images read MN-major) =================
        if (tid == 0) {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
            mma6(TX, [&](int i) { return tc::smem_desc(base + SM::A + i * (NCH * SLAB) + s * SLAB + kk * 32, 16, 1024, tc::LAYOUT_SW128); },
                 [&](int i) { return tc::smem_desc(base + SM::w2 + i * (D * D * 2) + (4 * s + kk) * 2048, D * 128, 1024, tc::LAYOUT_SW128); },
                 IDESC_ND_BT, (s | kk) != 0);
        }
      }
      mma_done();
      // ================= E3 / G4 =================
#pragma unroll
      for (int s = 0; s < NCH; ++s) {
        float x[16];
        tc::tmem_ld16(TX + tlane + (uint32_t)(64 * s + 16 * g), x);
#pragma unroll
        for (int k = 0; k < 16; ++k) x[k] *= ds[s][k];
        if (valid) {
          float4* dst = reinterpret_cast<float4*>(a.abar + (size_t)(e0 + row) * D + 64 * s + 16 * g);
#pragma unroll
          for (int k4 = 0; k4 < 4; ++k4) dst[k4] = make_float4(x[4 * k4], x[4 * k4 + 1], x[4 * k4 + 2], x[4 * k4 + 3]);
        }
        store_split16(Aop + s * SLAB, so0, so1, x);
        operands_ready();
        if (tid == 0) {
          // B = the G1 images [channel][32] read MN-major (N = 32, K = channel): K-direction 8-channel group stride
          // (LBO) 512 B, N-direction core-matrix stride (SBO) 128 B
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
            mma6(T4, [&](int i) { return tc::smem_desc(base + SM::A + i * (NCH * SLAB) + s * SLAB + kk * 32, 16, 1024, tc::LAYOUT_SW128); },
                 [&](int i) { return tc::smem_desc(base + SM::w13 + i * (D * K1 * 2) + (4 * s + kk) * 1024, 512, 128, tc::LAYOUT_NONE); },
                 IDESC_N32_BT, (s | kk) != 0);
        }
      }
    }
    // ================= GS: segmented sum of the slabs =================
    const int R = G.R;
    if (R <= MAX_SEG) {
      if (tid == 0) {
        constexpr int IS[3] = {2, 1, 0};
#pragma unroll
        for (int j = 0; j < TE / 16; ++j)
#pragma unroll
          for (int t = 0; t < 3; ++t)
            tc::mma_bf16(TS, tc::smem_desc(base + SM::A + IS[t] * (NCH * SLAB) + j * 2048, SLAB, 1024, tc::LAYOUT_SW128),
                         tc::smem_desc(base + SM::sel + j * 256, 128, 2048, tc::LAYOUT_NONE), IDESC_SEG, (j | t) != 0);
      }
      mma_done();
      if (g == 0) {
        float acc[16];
        tc::tmem_ld16(TS + tlane, acc);
#pragma unroll
        for (int r = 0; r < MAX_SEG; ++r)
          if (r < R) G.dst[r][row] = acc[r];
      }
    } else {
      if (BWD) mma_done();  // G4
      if (tid < D) segmented_store_x3(Aop, recv_s, a.rowptr, e0, tile, BWD ? a.Pbar : a.m, a.head, a.tail, tid);
    }
    if (BWD && g == 1) {
      // ================= E4 =================
      float eb[16], tb[16];
      tc::tmem_ld16(T4 + tlane, eb);
      tc::tmem_ld16(T4 + tlane + 16u, tb);
      if (valid) {
        if (a.tbar) {
          float4* dst = reinterpret_cast<float4*>(a.tbar + (size_t)(e0 + row) * 16);
#pragma unroll
          for (int k4 = 0; k4 < 4; ++k4) dst[k4] = make_float4(tb[4 * k4], tb[4 * k4 + 1], tb[4 * k4 + 2], tb[4 * k4 + 3]);
        }
        const float r = r_s[row], u = u_s[row], du = du_s[row];
        float part = 0.f;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          if (k < a.n_rbf) {
            float gk, dg;
            rbf_f(r, a.r_cut, a.n_rbf, k, gk, dg);
            part = fmaf(eb[k], fmaf(du, gk, u * dg), part);
          }
        }
        const float ubar = a.alpha * ((ubar_s[row] + ubar_s[TE + row]) + (ubar_s[2 * TE + row] + ubar_s[3 * TE + row]));
        a.rbar[e0 + row] += fmaf(ubar, du, part);
      }
    }
    // the next tile overwrites the metadata, the selector and the operand slabs, and its G1 region X
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
  }
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
