// MLIP_BF16 path of the fused edge kernels (steps A6, A7 and the edge part of A10) on the sm_100a
// tensor cores: bf16 operands, fp32 accumulation in TMEM.
//
// A persistent CTA (one per SM) keeps the bf16 image of W2 (and the small W1c images) resident in
// shared memory and walks over tiles of 128 consecutive receiver-sorted edges. Per tile:
//   G1  D1[edge, c]  = e_hat[edge, 0:16] . W1c^T                       tcgen05.mma  M128 N=d K16
//   E1  a = D1 + P_i + Q_j ; s = SiLU(a) -> bf16 S tile (the gathered Q rows are overwritten in
//       place); backward keeps SiLU'(a) in D1 (tcgen05.st)
//   G2  D2[edge, c]  = S . W2^T                                          K-major W2 image
//   E2  forward : phi = SiLU(D2 + b2), alpha u_e phi -> S tile, segmented column sums -> m_i
//       backward: pbar = alpha u_e mbar_i SiLU'(D2 + b2) -> S tile; ubar_e = alpha <mbar_i, phi_e>
//   G3  D3[edge, c']  = pbar . W2    (the SAME W2 image read as an MN-major operand)
//   E3  abar = D3 * SiLU'(a) -> S tile -> (i) one linear bulk copy to the spill buffer (read back
//       through rev[] by k_gather_rev_bf16), (ii) segmented column sums -> Pbar_i, (iii) G4
//   G4  D4[edge, k]  = abar . W1c   (ebar)                               N = 16
//   E4  rbar_e += ubar_e u' + sum_k ebar_k (u' g_k + u g'_k)
// Each thread owns one edge row (TMEM lane) and half of the channels. Segments that straddle
// tiles go through per-tile head/tail rows and k_segment_fixup_bf16: no floating-point atomics.
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"
#include "tc_ptx.cuh"

namespace {
constexpr int TE = 128;  // edges per tile = MMA M

template <int D>
struct ES {  // shared-memory carve-up, offsets from a 1024-byte aligned base
  static constexpr uint32_t w2 = 0;                          // [D x D] bf16, K-major SW128 image
  static constexpr uint32_t s = w2 + D * D * 2;              // [128 x D] bf16, K-major SW128
  static constexpr uint32_t w1cT = s + TE * D * 2;           // [16 x D] bf16, K-major SW128
  static constexpr uint32_t w1c = w1cT + 16 * D * 2;         // [D x 16] bf16, K-major no swizzle
  static constexpr uint32_t ehat = w1c + D * 16 * 2;         // [128 x 16] bf16, K-major no swizzle
  static constexpr uint32_t b2 = ehat + TE * 16 * 2;         // [D] fp32
  static constexpr uint32_t recv = b2 + D * 4;               // [128] int
  static constexpr uint32_t u = recv + TE * 4;               // [128] fp32
  static constexpr uint32_t du = u + TE * 4;
  static constexpr uint32_t r = du + TE * 4;
  static constexpr uint32_t ubar = r + TE * 4;               // [2][128] fp32
  static constexpr uint32_t bar = ubar + 2 * TE * 4;         // mbarrier
  static constexpr uint32_t slot = bar + 8;                  // TMEM base address
  static constexpr uint32_t bytes = slot + 8 + 1024;         // + alignment slack
  static constexpr int tmem_cols = 2 * D;                    // D1 | D2 (D3, D4 alias D2)
};

// Column sums of the bf16 S tile over runs of equal receiver (thread = channel). Complete segments
// go to out[recv], segments continuing from an earlier tile to head[tile], segments continuing
// into a later tile to tail[tile].
template <int D>
__device__ __forceinline__ void segmented_store_bf16(const unsigned char* __restrict__ S, const int* __restrict__ recv_s,
                                                     const int32_t* __restrict__ rowptr, int64_t e0, int64_t tile,
                                                     float* __restrict__ out, float* __restrict__ head,
                                                     float* __restrict__ tail, int c) {
  int cur = recv_s[0];
  float sum = 0.f;
  const uint32_t coff = (uint32_t)((c >> 6) * TE * 128 + (c & 7) * 2);
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
      const unsigned short v = *reinterpret_cast<const unsigned short*>(S + coff + e * 128 + ((cc ^ (e & 7)) << 4));
      sum += __uint_as_float((uint32_t)v << 16);
    }
  }
}

template <int D, bool BWD>
__global__ void __launch_bounds__(256, 1) k_edge_bf16(EdgeArgs a, int64_t n_tiles) {
  extern __shared__ unsigned char smem_raw[];
  using SM = ES<D>;
  const uint32_t base = (tc::smem_u32(smem_raw) + 1023u) & ~1023u;
  unsigned char* gen = smem_raw + (base - tc::smem_u32(smem_raw));
  unsigned char* S = gen + SM::s;
  float* b2_s = reinterpret_cast<float*>(gen + SM::b2);
  int* recv_s = reinterpret_cast<int*>(gen + SM::recv);
  float* u_s = reinterpret_cast<float*>(gen + SM::u);
  float* du_s = reinterpret_cast<float*>(gen + SM::du);
  float* r_s = reinterpret_cast<float*>(gen + SM::r);
  float* ubar_s = reinterpret_cast<float*>(gen + SM::ubar);
  uint32_t* slot = reinterpret_cast<uint32_t*>(gen + SM::slot);
  const uint32_t bar = base + SM::bar;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int q = warp & 3, hf = warp >> 2;
  const int row = q * 32 + lane;

  // ---- one-time setup: resident weight images, barrier, TMEM ----
  {
    const uint4* src = reinterpret_cast<const uint4*>(a.W2img);
    uint4* dst = reinterpret_cast<uint4*>(gen + SM::w2);
    for (int i = tid; i < D * D * 2 / 16; i += 256) dst[i] = src[i];
    src = reinterpret_cast<const uint4*>(a.W1cimg);
    dst = reinterpret_cast<uint4*>(gen + SM::w1c);
    for (int i = tid; i < D * 16 * 2 / 16; i += 256) dst[i] = src[i];
    src = reinterpret_cast<const uint4*>(a.W1cTimg);
    dst = reinterpret_cast<uint4*>(gen + SM::w1cT);
    for (int i = tid; i < 16 * D * 2 / 16; i += 256) dst[i] = src[i];
    for (int i = tid; i < D; i += 256) b2_s[i] = a.b2[i];
  }
  if (tid == 0) {
    tc::mbar_init(bar, 1);
    tc::fence_mbar_init();
  }
  if (warp == 0) tc::tmem_alloc<SM::tmem_cols>(slot);
  tc::fence_proxy_async();
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *slot;
  const uint32_t tlane = tmem + ((uint32_t)(q * 32) << 16);
  uint32_t phase = 0;

  constexpr uint32_t IDESC_ND = tc::idesc_bf16(128, D, 0, 0);     // K-major A and B, N = D
  constexpr uint32_t IDESC_ND_BT = tc::idesc_bf16(128, D, 0, 1);  // B read MN-major
  constexpr uint32_t IDESC_N16 = tc::idesc_bf16(128, 16, 0, 0);

  for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int64_t e0 = tile * TE;

    // ---- tile metadata, edge features (A6) and the sender-row gather into the S tile ----
    if (tid < TE) {
      const int64_t e = e0 + tid;
      int rc = -1;
      float r = 0.f, u = 0.f, du = 0.f;
      if (e < a.E) {
        rc = a.recv[e]; r = a.rvec[e].w;
        envelope_f(r, a.r_cut, u, du);
      }
      recv_s[tid] = rc; u_s[tid] = u; du_s[tid] = du; r_s[tid] = r;
      uint32_t pk[8];
#pragma unroll
      for (int k = 0; k < 16; k += 2) {
        float g0 = 0.f, g1 = 0.f, dg;
        if (e < a.E && k < a.n_rbf) rbf_f(r, a.r_cut, a.n_rbf, k, g0, dg);
        if (e < a.E && k + 1 < a.n_rbf) rbf_f(r, a.r_cut, a.n_rbf, k + 1, g1, dg);
        pk[k >> 1] = tc::pack_bf16(u * g0, u * g1);
      }
      // K-major, no swizzle: 8x8 core matrices of 128 B; (row, k) -> (row/8)*256 + (k/8)*128 + (row%8)*16
      unsigned char* dst = gen + SM::ehat + (tid >> 3) * 256 + (tid & 7) * 16;
      *reinterpret_cast<uint4*>(dst) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
      *reinterpret_cast<uint4*>(dst + 128) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
    }
#pragma unroll 4
    for (int i = 0; i < TE / 8; ++i) {
      const int rw = warp + 8 * i;
      const int64_t e = e0 + rw;
      if (lane < D / 8) {
        const uint32_t off = tc::sw128_chunk_off(TE, rw, lane);
        if (e < a.E) {
          const int sd = a.send[e];
          tc::cp_async16(base + SM::s + off, a.Qbf + (size_t)sd * D + lane * 8);
        } else {
          *reinterpret_cast<uint4*>(S + off) = make_uint4(0u, 0u, 0u, 0u);
        }
      }
    }
    tc::cp_async_commit();
    tc::cp_async_wait<0>();
    tc::fence_proxy_async();
    __syncthreads();

    // ---- G1: D1 = e_hat . W1c^T ----
    if (tid == 0) {
      tc::fence_after_sync();
      const uint64_t ad = tc::smem_desc(base + SM::ehat, 128, 256, tc::LAYOUT_NONE);
      const uint64_t bd = tc::smem_desc(base + SM::w1c, 128, 256, tc::LAYOUT_NONE);
      tc::mma_bf16(tmem, ad, bd, IDESC_ND, false);
      tc::mma_commit(bar);
    }
    tc::mbar_wait(bar, phase); phase ^= 1;
    tc::fence_after_sync();

    // ---- E1: a = D1 + P_i + Q_j ; s = SiLU(a) ----
    const int rc = recv_s[row];
    const bool valid = rc >= 0;
    {
      const float* Prow = a.P + (size_t)(valid ? rc : 0) * a.ldp;
#pragma unroll 1
      for (int c0 = hf * (D / 2); c0 < (hf + 1) * (D / 2); c0 += 32) {
        float acc[32];
        tc::tmem_ld32(tlane + (uint32_t)c0, acc);
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          unsigned char* sp = S + tc::sw128_chunk_off(TE, row, (c0 >> 3) + g);
          const uint4 qv = *reinterpret_cast<const uint4*>(sp);
          uint4 outv = make_uint4(0u, 0u, 0u, 0u);
          if (valid) {
            const float4 p0 = *reinterpret_cast<const float4*>(Prow + c0 + 8 * g);
            const float4 p1 = *reinterpret_cast<const float4*>(Prow + c0 + 8 * g + 4);
            const float pv[8] = {p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w};
            const float qf[8] = {tc::bf16_lo(qv.x), tc::bf16_hi(qv.x), tc::bf16_lo(qv.y), tc::bf16_hi(qv.y),
                                 tc::bf16_lo(qv.z), tc::bf16_hi(qv.z), tc::bf16_lo(qv.w), tc::bf16_hi(qv.w)};
            float sv[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              float ds;
              silu_both_f(acc[8 * g + j] + pv[j] + qf[j], sv[j], ds);
              acc[8 * g + j] = ds;
            }
            outv = make_uint4(tc::pack_bf16(sv[0], sv[1]), tc::pack_bf16(sv[2], sv[3]), tc::pack_bf16(sv[4], sv[5]),
                              tc::pack_bf16(sv[6], sv[7]));
          }
          *reinterpret_cast<uint4*>(sp) = outv;
        }
        if (BWD) tc::tmem_st32(tlane + (uint32_t)c0, acc);  // keep SiLU'(a) for E3
      }
      if (BWD) tc::tmem_wait_st();
    }
    tc::fence_proxy_async();
    tc::fence_before_sync();
    __syncthreads();

    // ---- G2: D2 = S . W2^T ----
    if (tid == 0) {
      tc::fence_after_sync();
#pragma unroll
      for (int kk = 0; kk < D / 16; ++kk) {
        const uint64_t ad = tc::smem_desc(base + SM::s + (kk >> 2) * (TE * 128) + (kk & 3) * 32, 16, 1024, tc::LAYOUT_SW128);
        const uint64_t bd = tc::smem_desc(base + SM::w2 + (kk >> 2) * (D * 128) + (kk & 3) * 32, 16, 1024, tc::LAYOUT_SW128);
        tc::mma_bf16(tmem + D, ad, bd, IDESC_ND, kk != 0);
      }
      tc::mma_commit(bar);
    }
    tc::mbar_wait(bar, phase); phase ^= 1;
    tc::fence_after_sync();

    if (!BWD) {
      // ---- E2 forward: alpha u_e SiLU(p) -> S tile, then segmented column sums ----
      const float w = valid ? a.alpha * u_s[row] : 0.f;
#pragma unroll 1
      for (int c0 = hf * (D / 2); c0 < (hf + 1) * (D / 2); c0 += 32) {
        float acc[32];
        tc::tmem_ld32(tlane + (uint32_t)(D + c0), acc);
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          float v[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) v[j] = w * silu_f(acc[8 * g + j] + b2_s[c0 + 8 * g + j]);
          *reinterpret_cast<uint4*>(S + tc::sw128_chunk_off(TE, row, (c0 >> 3) + g)) =
              make_uint4(tc::pack_bf16(v[0], v[1]), tc::pack_bf16(v[2], v[3]), tc::pack_bf16(v[4], v[5]),
                         tc::pack_bf16(v[6], v[7]));
        }
      }
      tc::fence_before_sync();
      __syncthreads();
      if (tid < D) segmented_store_bf16<D>(S, recv_s, a.rowptr, e0, tile, a.m, a.head, a.tail, tid);
      __syncthreads();
      continue;
    }

    // ---- E2 backward: pbar = alpha u mbar_i SiLU'(p) ; ubar_e = alpha <mbar_i, phi_e> ----
    {
      const float au = valid ? a.alpha * u_s[row] : 0.f;
      const float* mrow = a.mbar + (size_t)(valid ? rc : 0) * D;
      float ub = 0.f;
#pragma unroll 1
      for (int c0 = hf * (D / 2); c0 < (hf + 1) * (D / 2); c0 += 32) {
        float acc[32];
        tc::tmem_ld32(tlane + (uint32_t)(D + c0), acc);
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          float v[8];
          float mb[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
          if (valid) {
            const float4 m0 = *reinterpret_cast<const float4*>(mrow + c0 + 8 * g);
            const float4 m1 = *reinterpret_cast<const float4*>(mrow + c0 + 8 * g + 4);
            mb[0] = m0.x; mb[1] = m0.y; mb[2] = m0.z; mb[3] = m0.w; mb[4] = m1.x; mb[5] = m1.y; mb[6] = m1.z; mb[7] = m1.w;
          }
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            float phi, dphi;
            silu_both_f(acc[8 * g + j] + b2_s[c0 + 8 * g + j], phi, dphi);
            ub = fmaf(mb[j], phi, ub);
            v[j] = au * mb[j] * dphi;
          }
          *reinterpret_cast<uint4*>(S + tc::sw128_chunk_off(TE, row, (c0 >> 3) + g)) =
              make_uint4(tc::pack_bf16(v[0], v[1]), tc::pack_bf16(v[2], v[3]), tc::pack_bf16(v[4], v[5]),
                         tc::pack_bf16(v[6], v[7]));
        }
      }
      ubar_s[hf * TE + row] = ub;
    }
    tc::fence_proxy_async();
    tc::fence_before_sync();
    __syncthreads();

    // ---- G3: D3 = pbar . W2 (W2 image as MN-major B: LBO = slab stride, 16 k-rows = 2 KB) ----
    if (tid == 0) {
      tc::fence_after_sync();
#pragma unroll
      for (int kk = 0; kk < D / 16; ++kk) {
        const uint64_t ad = tc::smem_desc(base + SM::s + (kk >> 2) * (TE * 128) + (kk & 3) * 32, 16, 1024, tc::LAYOUT_SW128);
        const uint64_t bd = tc::smem_desc(base + SM::w2 + kk * 2048, D * 128, 1024, tc::LAYOUT_SW128);
        tc::mma_bf16(tmem + D, ad, bd, IDESC_ND_BT, kk != 0);
      }
      tc::mma_commit(bar);
    }
    tc::mbar_wait(bar, phase); phase ^= 1;
    tc::fence_after_sync();

    // ---- E3: abar = sbar * SiLU'(a) -> S tile ----
#pragma unroll 1
    for (int c0 = hf * (D / 2); c0 < (hf + 1) * (D / 2); c0 += 32) {
      float sb[32], ds[32];
      tc::tmem_ld32(tlane + (uint32_t)(D + c0), sb);
      tc::tmem_ld32(tlane + (uint32_t)c0, ds);
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        float v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = valid ? sb[8 * g + j] * ds[8 * g + j] : 0.f;
        *reinterpret_cast<uint4*>(S + tc::sw128_chunk_off(TE, row, (c0 >> 3) + g)) =
            make_uint4(tc::pack_bf16(v[0], v[1]), tc::pack_bf16(v[2], v[3]), tc::pack_bf16(v[4], v[5]),
                       tc::pack_bf16(v[6], v[7]));
      }
    }
    tc::fence_proxy_async();
    tc::fence_before_sync();
    __syncthreads();

    // ---- spill (bulk copy), G4: D4 = abar . W1c, segmented column sums -> Pbar ----
    if (tid == 0) {
      tc::fence_after_sync();
      tc::bulk_s2g(a.abar_bf + (size_t)tile * TE * D, base + SM::s, TE * D * 2);
      tc::bulk_commit();
#pragma unroll
      for (int kk = 0; kk < D / 16; ++kk) {
        const uint64_t ad = tc::smem_desc(base + SM::s + (kk >> 2) * (TE * 128) + (kk & 3) * 32, 16, 1024, tc::LAYOUT_SW128);
        const uint64_t bd = tc::smem_desc(base + SM::w1cT + (kk >> 2) * (16 * 128) + (kk & 3) * 32, 16, 1024, tc::LAYOUT_SW128);
        tc::mma_bf16(tmem + D, ad, bd, IDESC_N16, kk != 0);
      }
      tc::mma_commit(bar);
    }
    if (tid < D) segmented_store_bf16<D>(S, recv_s, a.rowptr, e0, tile, a.Pbar, a.head, a.tail, tid);
    tc::mbar_wait(bar, phase); phase ^= 1;
    tc::fence_after_sync();

    // ---- E4: rbar_e += ubar u' + sum_k ebar_k (u' g_k + u g'_k) ----
    if (warp < 4) {
      float eb[16];
      tc::tmem_ld16(tlane + (uint32_t)D, eb);
      const float r = r_s[row], u = u_s[row], du = du_s[row];
      float part = 0.f;
#pragma unroll
      for (int k = 0; k < 16; ++k) {
        if (k < a.n_rbf) {
          float g, dg;
          rbf_f(r, a.r_cut, a.n_rbf, k, g, dg);
          part = fmaf(eb[k], fmaf(du, g, u * dg), part);
        }
      }
      const float ubar = a.alpha * (ubar_s[row] + ubar_s[TE + row]);
      if (valid) a.rbar[e0 + row] += fmaf(ubar, du, part);
    }
    if (tid == 0) tc::bulk_wait_read0();  // the spill has finished reading the S tile
    tc::fence_before_sync();
    __syncthreads();
  }

  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<SM::tmem_cols>(tmem);
}

// out[i] = tail[t] + head[t+1] + ... for the segment that starts in tile t and continues beyond it
__global__ void k_segment_fixup_bf16(int64_t E, int D, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ recv,
                                     const float* __restrict__ head, const float* __restrict__ tail,
                                     float* __restrict__ out) {
  const int64_t t = blockIdx.x;
  const int64_t e0 = t * TE, e1 = e0 + TE;
  if (e1 >= E) return;
  const int i = recv[e1 - 1];
  const int64_t s0 = rowptr[i], s1 = rowptr[i + 1];
  if (!(s1 > e1 && s0 >= e0)) return;
  for (int c = threadIdx.x; c < D; c += blockDim.x) {
    float sum = tail[(size_t)t * D + c];
    for (int64_t t2 = t + 1; t2 * TE < s1; ++t2) sum += head[(size_t)t2 * D + c];
    out[(size_t)i * D + c] = sum;
  }
}

// Qbar_j = sum_{e in in(j)} abar[rev[e]]; abar rows live in the swizzled tile images written by E3
template <int D>
__global__ void __launch_bounds__(256) k_gather_rev_bf16(int64_t n, const int32_t* __restrict__ rowptr,
                                                         const int32_t* __restrict__ rev,
                                                         const __nv_bfloat16* __restrict__ abar, float* __restrict__ Qbar) {
  constexpr int CH = D / 8;        // 16-byte chunks per row
  constexpr int NSUB = 32 / CH;    // edges handled concurrently by one warp
  const int lane = threadIdx.x & 31;
  const int64_t j = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (j >= n) return;
  const int ch = lane % CH, sub = lane / CH;
  const int lo = rowptr[j], hi = rowptr[j + 1];
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  const unsigned char* base = reinterpret_cast<const unsigned char*>(abar);
  for (int e = lo + sub; e < hi; e += NSUB) {
    const int re = rev[e];
    const int t = re >> 7, rw = re & 127;
    const uint4 v = *reinterpret_cast<const uint4*>(base + (size_t)t * TE * D * 2 + tc::sw128_chunk_off(TE, rw, ch));
    acc[0] += tc::bf16_lo(v.x); acc[1] += tc::bf16_hi(v.x); acc[2] += tc::bf16_lo(v.y); acc[3] += tc::bf16_hi(v.y);
    acc[4] += tc::bf16_lo(v.z); acc[5] += tc::bf16_hi(v.z); acc[6] += tc::bf16_lo(v.w); acc[7] += tc::bf16_hi(v.w);
  }
  if (NSUB > 1) {
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], 16);
  }
  if (sub == 0) {
    float* dst = Qbar + (size_t)j * D + ch * 8;
    *reinterpret_cast<float4*>(dst) = make_float4(acc[0], acc[1], acc[2], acc[3]);
    *reinterpret_cast<float4*>(dst + 4) = make_float4(acc[4], acc[5], acc[6], acc[7]);
  }
}

template <int D>
int launch_edge(mlip_ctx* ctx, const EdgeArgs& a, bool bwd) {
  const int64_t tiles = (a.E + TE - 1) / TE;
  if (tiles == 0) return MLIP_OK;
  const size_t smem = ES<D>::bytes;
  const unsigned grid = (unsigned)(tiles < ctx->num_sms ? tiles : ctx->num_sms);
  if (bwd) {
    MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_edge_bf16<D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_edge_bf16<D, true><<<grid, 256, smem, ctx->stream>>>(a, tiles);
  } else {
    MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_edge_bf16<D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_edge_bf16<D, false><<<grid, 256, smem, ctx->stream>>>(a, tiles);
  }
  k_segment_fixup_bf16<<<(unsigned)tiles, D < 256 ? D : 256, 0, ctx->stream>>>(a.E, D, a.rowptr, a.recv, a.head, a.tail,
                                                                               bwd ? a.Pbar : a.m);
  ctx->launches += 2;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
}  // namespace

int64_t mlip_edge_bf16_tiles(int64_t E) { return (E + TE - 1) / TE; }

int mlip_edge_forward_bf16(mlip_ctx* ctx, int d, const EdgeArgs& a) {
  if (d == 256) return launch_edge<256>(ctx, a, false);
  if (d == 128) return launch_edge<128>(ctx, a, false);
  ctx->set_error("bf16 edge kernels need d = 128 or 256");
  return MLIP_ERR_UNSUPPORTED;
}
int mlip_edge_backward_bf16(mlip_ctx* ctx, int d, const EdgeArgs& a) {
  if (d == 256) return launch_edge<256>(ctx, a, true);
  if (d == 128) return launch_edge<128>(ctx, a, true);
  ctx->set_error("bf16 edge kernels need d = 128 or 256");
  return MLIP_ERR_UNSUPPORTED;
}
int mlip_gather_rev_bf16(mlip_ctx* ctx, int64_t n, int d, const int32_t* rowptr, const int32_t* rev,
                         const __nv_bfloat16* abar, float* Qbar) {
  if (n <= 0) return MLIP_OK;
  const unsigned grid = (unsigned)((n * 32 + 255) / 256);
  if (d == 256) k_gather_rev_bf16<256><<<grid, 256, 0, ctx->stream>>>(n, rowptr, rev, abar, Qbar);
  else if (d == 128) k_gather_rev_bf16<128><<<grid, 256, 0, ctx->stream>>>(n, rowptr, rev, abar, Qbar);
  else { ctx->set_error("bf16 gather needs d = 128 or 256"); return MLIP_ERR_UNSUPPORTED; }
  ctx->launches++;
  return MLIP_OK;
}
