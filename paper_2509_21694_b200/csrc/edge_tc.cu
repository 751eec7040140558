// Tensor-core path (precision MLIP_BF16) of the fused edge kernels: steps A6, A7 and the edge part
// of A10 on the sm_100a tensor cores. 16-bit operands, fp32 accumulation in TMEM.
//
// Operand type: IEEE half (f16), not bf16. Same tcgen05 rate and bytes, three more mantissa bits, and
// -- the reason -- the epilogues can then run in packed f16x2 arithmetic (HADD2/HFMA2, one
// instruction per two elements) straight from the accumulators to the next operand with no
// unpack/convert/pack sequence per element: the epilogues, not the MMAs, bound this kernel (MUFU:
// one tanh per element at 16/clk/SM = 4096 cycles per 128x256 tile pair of epilogues against 2048
// cycles of tcgen05 per GEMM). Range: |pre-activations| and |adjoints| must stay below 6.5e4.
//
// One persistent, warp-specialised CTA per SM walks over tiles of 128 consecutive receiver-sorted
// edges. The f16 image of W2 (and the small W1c image) stays resident in shared memory.
//   warps 0..15  epilogue: thread = (edge row, 16 of every 64 channels); TMEM -> registers -> SiLU ->
//                f16 operand slab in shared memory, chunk by chunk (64 channels = one SW128 slab)
//   warp 16      one thread issues every tcgen05.mma as soon as the slab it needs is published
//   warp 17      segment producer: receivers of the tile, the selector operand of the segmented sum,
//                and the per-tile staging of the receiver rows P_i (and mbar_i) in shared memory
//   warp 18      feature producer, up to two tiles ahead: edge metadata, envelope, radial basis (A6), the
//                f16 e_hat operand of G1
// Per tile (all factors 1/2 of the SiLU arguments are folded into the weight images, so that
// SiLU(2x) = x + x tanh(x) costs one MUFU and one FMA):
//   G1  X[edge, c]  = e_hat . (W1c/2)^T                                  M128 N=d K16
//   E1  a' = X + P'_i + Q'_j ; s = SiLU(2a') -> slab c/64 ; backward keeps 2 SiLU'(2a') in registers
//   G2  Y[edge, o] += s . (W2/2)^T      issued per 64-channel K slab while E1 works on the next one
//   E2  forward : phi = SiLU(2(Y + b2/2)) -> slabs (the weight alpha u_e rides in the selector of GS)
//       backward: pbar = alpha u_e mbar_i SiLU'(p) -> slabs ; ubar_e = alpha <mbar_i, phi_e>
//   G3  X[edge, i] += pbar . (W2/2)     (backward; the SAME W2 image read MN-major), per slab
//   E3  abar = X * 2 SiLU'(2a') -> slabs -> (i) bulk copy to the spill buffer (read back through
//       rev[] by k_gather_rev_tc), (ii) segmented sum, (iii) G4
//   GS  segmented sum over runs of equal receiver as an MMA: Yseg[channel, r] = slab^T . Sel with the
//       selector Sel[edge, r] = weight of edge if it belongs to receiver slot r (M = 128 channels,
//       N = 16 receivers, K = 128 edges); its result is m_i (forward) / Pbar_i (backward). Tiles with
//       more than 16 receivers take a shared-memory loop.
//   G4  ebar[edge, k] = abar . (W1c/2)  (N = 16, the W1c image read MN-major)
//   E4  rbar_e += ubar_e u' + sum_k 2 ebar_k (u' g_k + u g'_k)
// Segments that straddle tiles go through per-tile head/tail rows and k_segment_fixup_tc. The only
// reduction instruction is the one addition per edge and layer into rbar (E4), whose order is fixed by the
// launch order, so results are bitwise reproducible.
// Backward scheduling notes (from in-kernel clock64 timelines, profiles/r1e): G1 of the next tile is issued
// slab by slab as E3 publishes (X columns released), ahead of that slab's G4 / GS; the spill copies are only
// waited for once per tile, after that G1; the first layer runs with node_adjoint = false (no spill, no
// segmented sum) and with row_index = species (P, Q are S-row tables).
#include <cuda.h>
#include <string.h>
#include <cuda_fp16.h>
#include <type_traits>
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"
#include "tc_ptx.cuh"

namespace {
constexpr int TE = 128;          // edges per tile = MMA M
constexpr int N_EPI_WARPS = 16;  // 4 lane quarters x 4 column groups
constexpr int WARP_MMA = 16, WARP_SEG = 17, WARP_FEAT = 18, N_FEAT_WARPS = 1;
constexpr int N_THREADS = 19 * 32;
constexpr int SLOT_BYTES = TE * 128;  // one [128 x 64] f16 SW128 slab
constexpr int MAX_SEG = 16;           // receivers per tile handled by the selector MMA
constexpr int NSLOT = 8;              // receivers per tile whose P_i / mbar_i rows are staged in shared memory

template <bool BWD>
struct TileMeta {       // written by the feature producers, double buffered
  int recv[TE];         // local receiver (-1 beyond E)
  int send[TE];
  float w[TE];          // alpha * u(r_e)   (0 beyond E)
  float r[BWD ? TE : 1], u[BWD ? TE : 1], du[BWD ? TE : 1];
};
struct TileSeg {        // written by the segment producer, double buffered
  float* dst[MAX_SEG];  // where the sum of receiver slot r goes: out[rid] if its segment is complete inside the tile,
                        // head[tile] if it continues from an earlier tile, tail[tile] if it continues into a later one
  int rid[MAX_SEG];     // receivers of the tile in order of appearance
  int R;                // number of distinct receivers in the tile
  int pad[3];
  unsigned char slot[TE];  // receiver slot of every edge row (valid when R <= NSLOT)
};

template <int D, bool BWD>
struct ES {  // shared-memory carve-up, offsets from a 1024-byte aligned base
  static constexpr int NCH = D / 64;
  static constexpr uint32_t w2 = 0;                                   // [D x D] f16, K-major SW128 image of W2/2
  static constexpr uint32_t ring = w2 + D * D * 2;                    // NCH slabs [128 x 64] f16, K-major SW128
  static constexpr uint32_t w1c = ring + NCH * SLOT_BYTES;            // [D x 16] f16, K-major no swizzle (W1c/2)
  static constexpr uint32_t ehat = w1c + D * 16 * 2;                  // [128 x 16] f16, K-major no swizzle
  static constexpr uint32_t sel = ehat + TE * 16 * 2;                 // [16 x 128] f16, K-major no swizzle
  static constexpr uint32_t ptile = sel + MAX_SEG * TE * 2;           // [NSLOT x D] f16: P'_i of the tile's receivers
  static constexpr uint32_t mtile = ptile + NSLOT * D * 2;            // [NSLOT x D] f16: mbar_i (backward)
  static constexpr uint32_t b2 = mtile + (BWD ? NSLOT * D * 2 : 0);   // [D] f16 (b2/2)
  static constexpr uint32_t meta = b2 + D * 2;                        // TileMeta[2]
  static constexpr uint32_t seg = meta + 2 * sizeof(TileMeta<BWD>);   // TileSeg[2]
  static constexpr uint32_t ubar = seg + 2 * sizeof(TileSeg);         // [4][128] fp32 (backward)
  static constexpr uint32_t bars = ubar + (BWD ? 4 * TE * 4 : 0);     // mbarriers
  static constexpr uint32_t slot = bars + 32 * 8;                     // TMEM base address
  static constexpr uint32_t bytes = slot + 16 + 1024;                 // + alignment slack
  static constexpr int tmem_cols = 2 * D;                             // X | Y
  static_assert(bytes <= 232448, "shared memory budget of one SM exceeded");
};

// barrier indices
enum { B_META_FULL = 0, B_META_EMPTY = 2, B_EHAT_FULL = 4, B_SEL_FULL = 5, B_D1_FULL = 6, B_D2_FULL = 7,
       B_D3_FULL = 8, B_SEG_FULL = 9, B_X_FREE = 11, B_P_FULL = 12, B_P_FREE = 13,
       B_MB_FULL = 14, B_MB_FREE = 15, B_D2B_FULL = 16, B_D3B_FULL = 17, B_S_READY = 18 /* .. +NCH */,
       B_SPILL_S = 22 /* .. +NCH: slab s of the previous tile has been read by its spill copy */ };

constexpr uint32_t H2_ONE = 0x3C003C00u, H2_HALF = 0x38003800u, H2_NEG_ONE = 0xBC00BC00u, H2_NEG_HALF = 0xB800B800u;

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// read-only global load that keeps its place among the other asm volatile statements (prefetch distance)
__device__ __forceinline__ uint4 ldg_nc_v4(const void* p) {
  uint4 v;
  asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
// 32 contiguous bytes (one sector) per thread in ONE 256-bit request: half the L1 wavefronts of two 128-bit loads
__device__ __forceinline__ void ldg_nc_v8(const void* p, uint4& lo, uint4& hi) {
  asm volatile("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(lo.x), "=r"(lo.y), "=r"(lo.z), "=r"(lo.w), "=r"(hi.x), "=r"(hi.y), "=r"(hi.z), "=r"(hi.w)
               : "l"(p));
}
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// All 16 Gaussians g_k(r) = exp(-(r/Delta - k)^2 / 2) of one edge from THREE exponentials instead of sixteen (the
// producers share the MUFU of their SM partition with four epilogue warps): with t = r/Delta - 8,
// g_8 = exp(-t^2/2) and g_{8+-m} = g_{8+-(m-1)} exp(+-t) exp(1/2 - m). |t| <= 8, so every intermediate stays
// within e^+-32 and the product of at most 8 factors keeps fp32 accuracy (the result is rounded to f16).
__device__ __forceinline__ void gaussians16(float r_over_delta, float (&g)[16]) {
  constexpr float L2E = 1.4426950408889634f;
  const float t = r_over_delta - 8.0f;
  float ex;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ex) : "f"(-0.5f * L2E * t * t));
  g[8] = ex;
  float bp, bm;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(bp) : "f"(L2E * t));
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(bm) : "f"(-L2E * t));
  // exp(1/2 - m), m = 1..8
  constexpr float C[9] = {0.f, 0.60653065971263342f, 0.22313016014842982f, 0.082084998623898800f, 0.030197383422318501f,
                          0.011108996538242306f, 0.0040867714384640666f, 0.0015034391929775724f, 0.00055308437014783363f};
#pragma unroll
  for (int m = 1; m <= 7; ++m) g[8 + m] = g[8 + m - 1] * (bp * C[m]);
#pragma unroll
  for (int m = 1; m <= 8; ++m) g[8 - m] = g[8 - m + 1] * (bm * C[m]);
}
__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void tmem_ld16_nowait(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
}

template <int N>
__device__ __forceinline__ void tmem_ld_nowait(uint32_t taddr, uint32_t (&r)[N]) {
  static_assert(N == 4 || N == 8, "4 or 8 columns");
  if constexpr (N == 8)
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

// Shared-memory fallback of the segmented sum (tiles with more than MAX_SEG receivers): column sums
// of the f16 slabs over runs of equal receiver (thread = channel), each row weighted by wrow[e] when
// given. Complete segments go to out[recv], segments continuing from an earlier tile to head[tile],
// segments continuing into a later tile to tail[tile].
template <int D>
__device__ __forceinline__ void segmented_store_tc(const unsigned char* __restrict__ S, const int* __restrict__ recv_s,
                                                   const float* __restrict__ wrow, const int32_t* __restrict__ rowptr,
                                                   int64_t e0, int64_t tile, float* __restrict__ out,
                                                   float* __restrict__ head, float* __restrict__ tail, int c) {
  int cur = recv_s[0];
  float sum = 0.f;
  const uint32_t coff = (uint32_t)((c >> 6) * SLOT_BYTES + (c & 7) * 2);
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
      const __half v = *reinterpret_cast<const __half*>(S + coff + e * 128 + ((cc ^ (e & 7)) << 4));
      sum = fmaf(wrow ? wrow[e] : 1.0f, __half2float(v), sum);
    }
  }
}

template <int D, bool BWD>
__global__ void __launch_bounds__(N_THREADS, 1) k_edge_tc(EdgeArgs a, int64_t n_tiles_cap,
                                                          const __grid_constant__ CUtensorMap spill_map) {
  extern __shared__ unsigned char smem_raw[];
  // number of edges: by value, or read from the device in Verlet-skin mode (EdgeArgs::E_dyn; a.E is then the capacity)
  const int64_t n_edges = a.E_dyn ? (int64_t)__ldg(a.E_dyn) : a.E;
  const int64_t n_tiles = a.E_dyn ? (n_edges + TE - 1) / TE : n_tiles_cap;
  using SM = ES<D, BWD>;
  using Meta = TileMeta<BWD>;
  constexpr int NCH = SM::NCH;
  const uint32_t base = (tc::smem_u32(smem_raw) + 1023u) & ~1023u;
  unsigned char* gen = smem_raw + (base - tc::smem_u32(smem_raw));
  Meta* meta = reinterpret_cast<Meta*>(gen + SM::meta);
  TileSeg* seg = reinterpret_cast<TileSeg*>(gen + SM::seg);
  float* ubar_s = reinterpret_cast<float*>(gen + SM::ubar);
  uint32_t* slot = reinterpret_cast<uint32_t*>(gen + SM::slot);
  auto bar = [&](int i) -> uint32_t { return base + SM::bars + 8u * (uint32_t)i; };

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  // ---- one-time setup: resident weight images, barriers, TMEM ----
  {
    const uint4* src = reinterpret_cast<const uint4*>(a.W2img);
    uint4* dst = reinterpret_cast<uint4*>(gen + SM::w2);
    for (int i = tid; i < D * D * 2 / 16; i += N_THREADS) dst[i] = src[i];
    src = reinterpret_cast<const uint4*>(a.W1cimg);
    dst = reinterpret_cast<uint4*>(gen + SM::w1c);
    for (int i = tid; i < D * 16 * 2 / 16; i += N_THREADS) dst[i] = src[i];
    __half* b2h = reinterpret_cast<__half*>(gen + SM::b2);
    for (int i = tid; i < D; i += N_THREADS) b2h[i] = __float2half_rn(0.5f * a.b2[i]);
    // staged rows start finite: a stale slot is never read, but keep the buffers defined
    uint4* z = reinterpret_cast<uint4*>(gen + SM::ptile);
    for (int i = tid; i < (BWD ? 2 : 1) * NSLOT * D * 2 / 16; i += N_THREADS) z[i] = make_uint4(0u, 0u, 0u, 0u);
  }
  if (tid == 0) {
    tc::mbar_init(bar(B_META_FULL), N_FEAT_WARPS); tc::mbar_init(bar(B_META_FULL + 1), N_FEAT_WARPS);
    tc::mbar_init(bar(B_META_EMPTY), N_EPI_WARPS); tc::mbar_init(bar(B_META_EMPTY + 1), N_EPI_WARPS);
    tc::mbar_init(bar(B_EHAT_FULL), N_FEAT_WARPS); tc::mbar_init(bar(B_SEL_FULL), 1);
    tc::mbar_init(bar(B_D1_FULL), 1); tc::mbar_init(bar(B_D2_FULL), 1); tc::mbar_init(bar(B_D3_FULL), 1);
    tc::mbar_init(bar(B_SEG_FULL), 1); tc::mbar_init(bar(B_X_FREE), N_EPI_WARPS);
    for (int s = 0; s < NCH; ++s) tc::mbar_init(bar(B_SPILL_S + s), 1);
    tc::mbar_init(bar(B_P_FULL), 1); tc::mbar_init(bar(B_P_FREE), N_EPI_WARPS);
    tc::mbar_init(bar(B_MB_FULL), 1); tc::mbar_init(bar(B_MB_FREE), N_EPI_WARPS);
    tc::mbar_init(bar(B_D2B_FULL), 1); tc::mbar_init(bar(B_D3B_FULL), 1);
    for (int s = 0; s < NCH; ++s) tc::mbar_init(bar(B_S_READY + s), N_EPI_WARPS);
    tc::fence_mbar_init();
  }
  if (warp == 0) tc::tmem_alloc<SM::tmem_cols>(slot);
  tc::fence_proxy_async();
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *slot;
  const uint32_t TX = tmem, TY = tmem + D;  // accumulator regions: X = D1 / D3, Y = D2 / (segment sums, D4)

  if (blockIdx.x >= n_tiles) {
    // no tile for this CTA (only possible with E_dyn: the grid is sized from the capacity)
  } else if (warp >= WARP_FEAT) {
    // ============ feature producers: tile metadata (two tiles ahead) and the e_hat operand ============
    const float delta = a.r_cut / (float)(a.n_rbf - 1);
    const float inv_delta = 1.0f / delta;
    const float inv_rc = 1.0f / a.r_cut;
    constexpr int EPL = TE / (32 * N_FEAT_WARPS);  // edges per lane
    const int ebase = (warp - WARP_FEAT) * (TE / N_FEAT_WARPS) + lane;  // this lane's edges: ebase + 32 k
    int it = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
      const int b = it & 1;
      Meta& M = meta[b];
      const int64_t e0 = tile * TE;
      int rc[EPL], sd[EPL];
      float rr[EPL];
#pragma unroll
      for (int k = 0; k < EPL; ++k) {
        const int64_t ge = e0 + ebase + 32 * k;
        rc[k] = -1; sd[k] = 0; rr[k] = 0.f;
        if (ge < n_edges) { rc[k] = a.recv[ge]; sd[k] = a.send[ge]; rr[k] = a.rvec[ge].w; }
      }
      if (a.row_index) {  // M.send carries the ROW of the Q table: the sender itself, or its species in the first layer
#pragma unroll
        for (int k = 0; k < EPL; ++k)
          if (rc[k] >= 0) sd[k] = a.row_index[sd[k]];
      }
      tc::mbar_wait(bar(B_META_EMPTY + b), (uint32_t)(((it >> 1) & 1) ^ 1));
      uint32_t pk[EPL][8];
#pragma unroll
      for (int k = 0; k < EPL; ++k) {
        const int e = ebase + 32 * k;
        float u = 0.f, du = 0.f;
        if (rc[k] >= 0) {
          float sn, cs;
          __sincosf(3.14159265358979f * rr[k] * inv_rc, &sn, &cs);  // argument in [0, pi]
          u = 0.5f * (cs + 1.0f);
          du = -(1.5707963267948966f * inv_rc) * sn;
        }
        M.recv[e] = rc[k]; M.send[e] = sd[k]; M.w[e] = a.alpha * u;
        if (BWD) { M.r[e] = rr[k]; M.u[e] = u; M.du[e] = du; }
        float gk[16];
        gaussians16(rr[k] * inv_delta, gk);
#pragma unroll
        for (int j = 0; j < 16; j += 2)
          pk[k][j >> 1] = tc::pack_f16(j < a.n_rbf ? u * gk[j] : 0.f, j + 1 < a.n_rbf ? u * gk[j + 1] : 0.f);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_META_FULL + b));
      // e_hat operand of G1: K-major, no swizzle: (row, k) -> (row/8)*256 + (k/8)*128 + (row%8)*16 + (k%8)*2
      if (it > 0) tc::mbar_wait(bar(B_D1_FULL), (uint32_t)((it - 1) & 1));  // G1 of the previous tile has read it
#pragma unroll
      for (int k = 0; k < EPL; ++k) {
        const int e = ebase + 32 * k;
        unsigned char* dst = gen + SM::ehat + (e >> 3) * 256 + (e & 7) * 16;
        *reinterpret_cast<uint4*>(dst) = make_uint4(pk[k][0], pk[k][1], pk[k][2], pk[k][3]);
        *reinterpret_cast<uint4*>(dst + 128) = make_uint4(pk[k][4], pk[k][5], pk[k][6], pk[k][7]);
      }
      tc::fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_EHAT_FULL));
    }
  } else if (warp == WARP_SEG) {
    // ===== segment producer: receivers of the tile, staged P_i / mbar_i rows, selector operand of GS =====
    int it = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
      const int b = it & 1;
      TileSeg& G = seg[b];
      const int64_t e0 = tile * TE;
      int rc[4];
      uint32_t fm[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int e = lane + 32 * k;
        const int64_t ge = e0 + e;
        bool flag = false;
        rc[k] = -1;
        if (ge < n_edges) {
          rc[k] = a.recv[ge];
          flag = e == 0 || a.recv[ge - 1] != rc[k];
        }
        fm[k] = __ballot_sync(0xffffffffu, flag);
      }
      int rloc[4], cls[4];
      int before = 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        rloc[k] = before + __popc(fm[k] & (0xffffffffu >> (31 - lane))) - 1;
        cls[k] = -1;
        if (((fm[k] >> lane) & 1u) && rloc[k] < MAX_SEG) {
          const int64_t s0 = a.rowptr[rc[k]], s1 = a.rowptr[rc[k] + 1];
          cls[k] = (s0 >= e0 && s1 <= e0 + TE) ? 0 : (s0 < e0 ? 1 : 2);
        }
        before += __popc(fm[k]);
      }
      const int R = before;
      const bool fast = R <= NSLOT;
      // ---- receiver list, row slots and the P'_i rows: free once E1 of the previous tile is done ----
      if (it > 0) tc::mbar_wait(bar(B_P_FREE), (uint32_t)((it - 1) & 1));
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (cls[k] >= 0) {
          G.rid[rloc[k]] = rc[k];
          G.dst[rloc[k]] = cls[k] == 0 ? (BWD ? a.Pbar : a.m) + (size_t)rc[k] * D
                                       : (cls[k] == 1 ? a.head : a.tail) + (size_t)tile * D;
        }
        G.slot[lane + 32 * k] = (unsigned char)(rloc[k] < 0 ? 0 : (rloc[k] & 15));
      }
      if (lane == 0) G.R = R;
      __syncwarp();
      if (fast) {
        if (lane < D / 8) {  // one row = D/8 chunks of 16 bytes
          uint4 pr[NSLOT];
#pragma unroll
          for (int r = 0; r < NSLOT; ++r)
            if (r < R) pr[r] = ldg_nc_v4(a.Ph + (size_t)(a.row_index ? a.row_index[G.rid[r]] : G.rid[r]) * D + lane * 8);
#pragma unroll
          for (int r = 0; r < NSLOT; ++r)
            if (r < R) *reinterpret_cast<uint4*>(gen + SM::ptile + r * D * 2 + lane * 16) = pr[r];
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_P_FULL));
      if (BWD) {
        // ---- mbar_i rows: the buffer is free once E2 of the previous tile is done; the loads do not wait for it ----
        uint4 mr[NSLOT];
        if (fast && lane < D / 8) {
#pragma unroll
          for (int r = 0; r < NSLOT; ++r)
            if (r < R) mr[r] = ldg_nc_v4(a.mbar_h + (size_t)G.rid[r] * D + lane * 8);
        }
        if (it > 0) tc::mbar_wait(bar(B_MB_FREE), (uint32_t)((it - 1) & 1));
        if (fast && lane < D / 8) {
#pragma unroll
          for (int r = 0; r < NSLOT; ++r)
            if (r < R) *reinterpret_cast<uint4*>(gen + SM::mtile + r * D * 2 + lane * 16) = mr[r];
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(B_MB_FULL));
      }
      // ---- selector: the buffer is free once GS of the previous tile is done ----
      float wsel[4];
      if (!BWD) {
        tc::mbar_wait(bar(B_META_FULL + b), (uint32_t)((it >> 1) & 1));
#pragma unroll
        for (int k = 0; k < 4; ++k) wsel[k] = meta[b].w[lane + 32 * k];
      }
      if (it > 0) tc::mbar_wait(bar(B_SEG_FULL), (uint32_t)((it - 1) & 1));
      {
        uint4* z = reinterpret_cast<uint4*>(gen + SM::sel);
#pragma unroll
        for (int i = 0; i < MAX_SEG * TE * 2 / 16 / 32; ++i) z[lane + 32 * i] = make_uint4(0u, 0u, 0u, 0u);
      }
      __syncwarp();
      // Sel[r][e] = weight of edge e if it belongs to the r-th receiver of the tile; K-major (K = edge), no
      // swizzle: (r, e) -> (r/8)*2048 + (e/8)*128 + (r%8)*16 + (e%8)*2
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int e = lane + 32 * k;
        if (rc[k] >= 0 && rloc[k] < MAX_SEG)
          *reinterpret_cast<__half*>(gen + SM::sel + (rloc[k] >> 3) * 2048 + (e >> 3) * 128 + (rloc[k] & 7) * 16 + (e & 7) * 2) =
              __float2half_rn(BWD ? 1.0f : wsel[k]);
      }
      tc::fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_SEL_FULL));
    }
  } else if (warp == WARP_MMA) {
    // =========================== MMA issuer (one thread) ===========================
    if (lane == 0) {
      constexpr uint32_t IDESC_ND = tc::idesc_f16(128, D, 0, 0);     // K-major A and B, N = D
      constexpr uint32_t IDESC_ND_BT = tc::idesc_f16(128, D, 0, 1);  // B read MN-major
      // the last K slab of G2 / G3 is issued as two N halves with a commit each, so that the epilogue of
      // the first half of the columns starts while the tensor core finishes the second
      constexpr uint32_t IDESC_NH = tc::idesc_f16(128, D / 2, 0, 0);
      constexpr uint32_t IDESC_NH_BT = tc::idesc_f16(128, D / 2, 0, 1);
      constexpr uint32_t IDESC_N16_BT = tc::idesc_f16(128, 16, 0, 1);
      constexpr uint32_t IDESC_SEG = tc::idesc_f16(128, 16, 1, 0);   // A read MN-major (M = channel, K = edge)
      constexpr uint32_t IDESC_N64 = tc::idesc_f16(128, 64, 0, 0);   // G1 of the next tile, one 64-column slab at a time
      uint32_t srp = 0;  // bit s: parity of the next completion of S_READY[s]
      auto wait_slab = [&](int s) {
        tc::mbar_wait(bar(B_S_READY + s), (srp >> s) & 1u);
        srp ^= 1u << s;
        tc::fence_after_sync();
      };
      auto issue_g1 = [&](int jt) {  // G1 of this CTA's jt-th tile: needs its e_hat and region X released by tile jt-1
        tc::mbar_wait(bar(B_EHAT_FULL), (uint32_t)(jt & 1));
        tc::mbar_wait(bar(B_X_FREE), (uint32_t)((jt & 1) ^ 1));
        tc::fence_after_sync();
        tc::mma_bf16(TX, tc::smem_desc(base + SM::ehat, 128, 256, tc::LAYOUT_NONE),
                     tc::smem_desc(base + SM::w1c, 128, 256, tc::LAYOUT_NONE), IDESC_ND, false);
        tc::mma_commit(bar(B_D1_FULL));
      };
      int it = 0;
      issue_g1(0);
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int b = it & 1;
        const bool has_next = tile + gridDim.x < n_tiles;
        // the spill copies of the previous tile have been in flight since its E3; by now (G1 of this tile is issued) they
        // have read their slabs, so this wait does not hold up the MMA issue the way a wait inside the GS loop did
        if (BWD && it > 0) {
          tc::bulk_wait_read<0>();
#pragma unroll
          for (int s = 0; s < NCH; ++s) mbar_arrive(bar(B_SPILL_S + s));
        }
        // G2, one K slab at a time
#pragma unroll
        for (int s = 0; s < NCH; ++s) {
          wait_slab(s);
          if (s < NCH - 1) {
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
              tc::mma_f16_ts(TY, TX + (uint32_t)(64 * s + 16 * kk),  // A = s, written in place over X by E1
                             tc::smem_desc(base + SM::w2 + s * (D * 128) + kk * 32, 16, 1024, tc::LAYOUT_SW128), IDESC_ND,
                             (s | kk) != 0);
          } else {
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
#pragma unroll
              for (int kk = 0; kk < 4; ++kk)
                tc::mma_f16_ts(TY + (uint32_t)(hf * (D / 2)), TX + (uint32_t)(64 * s + 16 * kk),
                               tc::smem_desc(base + SM::w2 + s * (D * 128) + hf * (D / 2) * 128 + kk * 32, 16, 1024,
                                             tc::LAYOUT_SW128),
                               IDESC_NH, true);
              tc::mma_commit(bar(hf == 0 ? B_D2_FULL : B_D2B_FULL));
            }
          }
        }
        if (!BWD && has_next) issue_g1(it + 1);  // forward: X is dead after E1, run G1 of the next tile under E2
        if (BWD) {
          // G3: X = pbar . W2 (W2 image as MN-major B: LBO = slab stride, 16 k-rows = 2 KB)
#pragma unroll
          for (int s = 0; s < NCH; ++s) {
            wait_slab(s);
            if (s < NCH - 1) {
#pragma unroll
              for (int kk = 0; kk < 4; ++kk)
                tc::mma_f16_ts(TX, TY + (uint32_t)(64 * s + 16 * kk),  // A = pbar, written in place over Y by E2
                               tc::smem_desc(base + SM::w2 + (4 * s + kk) * 2048, D * 128, 1024, tc::LAYOUT_SW128),
                               IDESC_ND_BT, (s | kk) != 0);
            } else {
#pragma unroll
              for (int hf = 0; hf < 2; ++hf) {
#pragma unroll
                for (int kk = 0; kk < 4; ++kk)
                  tc::mma_f16_ts(TX + (uint32_t)(hf * (D / 2)), TY + (uint32_t)(64 * s + 16 * kk),
                                 tc::smem_desc(base + SM::w2 + (4 * s + kk) * 2048 + hf * (D / 128) * (D * 128), D * 128, 1024,
                                               tc::LAYOUT_SW128),
                                 IDESC_NH_BT, true);
                tc::mma_commit(bar(hf == 0 ? B_D3_FULL : B_D3B_FULL));
              }
            }
          }
        }
        tc::mbar_wait(bar(B_SEL_FULL), (uint32_t)(it & 1));
        const bool seg_mma = *reinterpret_cast<volatile int*>(&seg[b].R) <= MAX_SEG && (!BWD || a.node_adjoint);
#pragma unroll
        for (int s = 0; s < NCH; ++s) {
          wait_slab(s);
          if (BWD && has_next) {
            // G1 of the NEXT tile, slab by slab and ahead of this slab's G4 / GS: E3 has just published slab s, i.e. read the
            // last of the X columns of this slab, so they can take the next tile's e_hat . W1c^T now instead of after the whole of E3 (the backward
            // kernel used to start every tile waiting ~1 k cycles for G1)
            if (s == 0) { tc::mbar_wait(bar(B_EHAT_FULL), (uint32_t)((it + 1) & 1)); tc::fence_after_sync(); }
            tc::mma_bf16(TX + (uint32_t)(64 * s), tc::smem_desc(base + SM::ehat, 128, 256, tc::LAYOUT_NONE),
                         tc::smem_desc(base + SM::w1c + s * 2048, 128, 256, tc::LAYOUT_NONE), IDESC_N64, false);
            if (s == NCH - 1) tc::mma_commit(bar(B_D1_FULL));
          }
          if (BWD) {
            // ā slab -> ROW-MAJOR spill [edge][channel] by a tensor-map store (the copy engine undoes the 128-byte swizzle),
            // so that the sender-side gather reads 2 d contiguous bytes per reverse edge
            if (a.node_adjoint) tc::tma_store_2d(&spill_map, base + SM::ring + s * SLOT_BYTES, 64 * s, (int)(tile * TE));
            tc::bulk_commit();  // one bulk group per slab: a slab is released as soon as ITS copy has read it
            // G4: ebar/2 = abar . (W1c/2). B = the G1 image [channel][16] read MN-major (N = rbf index, K = channel),
            // no swizzle: N-direction core-matrix stride (SBO) 128 B, K-direction 8-channel group stride (LBO) 256 B
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
              tc::mma_bf16(TY + 32, tc::smem_desc(base + SM::ring + s * SLOT_BYTES + kk * 32, 16, 1024, tc::LAYOUT_SW128),
                           tc::smem_desc(base + SM::w1c + (4 * s + kk) * 512, 256, 128, tc::LAYOUT_NONE), IDESC_N16_BT,
                           (s | kk) != 0);
          }
          if ((s & 1) && seg_mma) {  // GS over the 128 channels of slabs s-1, s
#pragma unroll
            for (int j = 0; j < TE / 16; ++j)
              tc::mma_bf16(TY + 16 * (s >> 1),
                           tc::smem_desc(base + SM::ring + (s - 1) * SLOT_BYTES + j * 2048, SLOT_BYTES, 1024, tc::LAYOUT_SW128),
                           tc::smem_desc(base + SM::sel + j * 256, 128, 2048, tc::LAYOUT_NONE), IDESC_SEG, j != 0);
          }
        }
        tc::mma_commit(bar(B_SEG_FULL));
      }
      if (BWD) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
  } else {
    // =========================== epilogue warps ===========================
    const int q = warp & 3, g = warp >> 2;
    const int row = q * 32 + lane;
    const uint32_t tlane = (uint32_t)(q * 32) << 16;
    // byte offsets of this thread's two 16-byte chunks (channels 16g..16g+15 of a slab) inside a slab
    const uint32_t so0 = (uint32_t)(row * 128 + (((2 * g) ^ (row & 7)) << 4));
    const uint32_t so1 = (uint32_t)(row * 128 + (((2 * g + 1) ^ (row & 7)) << 4));
    unsigned char* ring = gen + SM::ring;
    const unsigned char* b2h = gen + SM::b2 + 32 * g;  // this thread's 16 channels of b2/2 inside a 64-channel block
    float* out = BWD ? a.Pbar : a.m;

    auto publish = [&](int s) {  // slab s written by this warp: visible to the async proxy, then signal
      tc::fence_proxy_async();
      tc::fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_S_READY + s));
    };
    // operand chunk kept in tensor memory: this thread's 16 f16 (8 columns) over the first half of the 16 fp32
    // accumulator columns it has just read; no proxy fence, so loads in flight are not waited for
    auto publish_tmem = [&](int s) {
      tc::tmem_wait_st();
      tc::fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_S_READY + s));
    };
    auto store_slab = [&](int s, const uint32_t (&v)[8]) {
      *reinterpret_cast<uint4*>(ring + s * SLOT_BYTES + so0) = make_uint4(v[0], v[1], v[2], v[3]);
      *reinterpret_cast<uint4*>(ring + s * SLOT_BYTES + so1) = make_uint4(v[4], v[5], v[6], v[7]);
    };

    // Read-out of a finished tile: segment sums out of Y (and E4). Deferred into E1 of the NEXT tile (after its first
    // slab is computed, before that slab is published and G2 starts to overwrite Y), so that the selector MMAs and
    // their completion latency hide under useful work instead of ending every tile with an idle wait.
    auto read_out = [&](int itp, int64_t tile, bool valid) {
      const int b = itp & 1;
      const uint32_t par = (uint32_t)(itp & 1);
      const Meta& M = meta[b];
      const TileSeg& G = seg[b];
      const int64_t e0 = tile * TE;
      const int R = G.R;
      tc::mbar_wait(bar(B_SEG_FULL), par);
      tc::fence_after_sync();
      if (BWD && !a.node_adjoint) {
        // first layer: no node-side adjoint wanted, only E4 below
      } else if (R <= MAX_SEG) {
        // Yseg: 16 columns (receiver slots) per 128 channels; warp group g reads 2 NCH of the 8 NCH columns
        constexpr int NR = 2 * NCH;
        const int h = (g * NR) >> 4, r0 = (g * NR) & 15;
        if (r0 < R) {
          uint32_t acc[NR];
          tmem_ld_nowait<NR>(TY + tlane + (uint32_t)(g * NR), acc);
          tc::tmem_wait_ld();
          const int pos = 128 * h + row;
#pragma unroll
          for (int r = 0; r < NR; ++r)
            if (r0 + r < R) G.dst[r0 + r][pos] = __uint_as_float(acc[r]);
        }
      } else {
        named_bar_sync(1, N_EPI_WARPS * 32);
        if (tid < D) segmented_store_tc<D>(ring, M.recv, BWD ? nullptr : M.w, a.rowptr, e0, tile, out, a.head, a.tail, tid);
        named_bar_sync(1, N_EPI_WARPS * 32);
      }
      // (column group 1: with the usual 3-4 receivers per tile only groups 0 and 2 have segment sums to read out above,
      // so E4 goes to a group that would otherwise idle here while the others wait for it at the next barrier)
      if (BWD && g == 1) {
        // ---- E4: rbar_e += ubar u' + sum_k ebar_k (u' g_k + u g'_k); G4 used the halved W1c image ----
        uint32_t eb[16];
        tmem_ld16_nowait(TY + tlane + 32u, eb);
        tc::tmem_wait_ld();
        // u' g_k + u g'_k = g_k (u' - 2 gamma u (r - k Delta)), g_k through ex2.approx as in the feature producers
        const float r = M.r[row], u = M.u[row], du = M.du[row];
        const float delta = a.r_cut / (float)(a.n_rbf - 1);
        const float gamma = 0.5f / (delta * delta);
        const float c1 = -2.0f * gamma * u;
        float gk[16];
        gaussians16(r / delta, gk);
        float part = 0.f;
#pragma unroll
        for (int k = 0; k < 16; ++k)
          if (k < a.n_rbf) part = fmaf(__uint_as_float(eb[k]), gk[k] * fmaf(c1, r - (float)k * delta, du), part);
        const float ubar = a.alpha * ((ubar_s[row] + ubar_s[TE + row]) + (ubar_s[2 * TE + row] + ubar_s[3 * TE + row]));
        // one addition per edge and layer, layers are separate launches: a fire-and-forget reduction is deterministic
        // and, unlike a read-modify-write, has no global-load latency inside E1 of the next tile
        if (valid) atomicAdd(a.rbar + e0 + row, fmaf(ubar, du, 2.0f * part));
      }
      tc::fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(B_META_EMPTY + b));
    };

    // row metadata and the first Q chunk of a tile are fetched while the previous tile drains
    tc::mbar_wait(bar(B_META_FULL), 0u);
    int rc = meta[0].recv[row];
    float w = meta[0].w[row];
    const __half* Qrow = a.Qh + (size_t)(rc >= 0 ? meta[0].send[row] : 0) * D + 16 * g;
    // Q'_j chunks of the row, fetched QD - 1 slabs ahead of their use (rolling buffer of QD)
    constexpr int QD = 3;
    uint4 qb[QD][2];
#pragma unroll
    for (int s = 0; s < QD - 1; ++s) ldg_nc_v8(Qrow + 64 * s, qb[s][0], qb[s][1]);

    int it = 0;
    bool valid_prev = false;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
      const int b = it & 1;
      const uint32_t par = (uint32_t)(it & 1);
      const Meta& M = meta[b];
      const TileSeg& G = seg[b];
      const int64_t e0 = tile * TE;
      const bool has_next = tile + gridDim.x < n_tiles;
      const bool valid = rc >= 0;

      // receiver rows of the tile: staged in shared memory (R <= NSLOT) or read from global memory
      tc::mbar_wait(bar(B_P_FULL), par);
      const int R = G.R;
      const bool fast = R <= NSLOT;
      const int myslot = G.slot[row];
      const unsigned char* prow = fast ? gen + SM::ptile + myslot * (D * 2) + 32 * g
                                       : reinterpret_cast<const unsigned char*>(
                                             a.Ph + (size_t)(valid ? (a.row_index ? a.row_index[rc] : rc) : 0) * D + 16 * g);

      // ---- E1: a' = X + P'_i + Q'_j ; s = a' + a' tanh(a') ----
      tc::mbar_wait(bar(B_D1_FULL), par);
      tc::fence_after_sync();
      // (the loop exists twice, for tiles whose receiver rows are staged in shared memory and for the others: a per-load
      // select between the two sources costs the staged path the registers and scoreboards of the global loads)
      auto e1_loop = [&](auto staged) {
      constexpr bool STAGED = decltype(staged)::value;
#pragma unroll
      for (int s = 0; s < NCH; ++s) {
        uint32_t acc[16];
        tmem_ld16_nowait(TX + tlane + (uint32_t)(64 * s + 16 * g), acc);
        const uint4 q0 = qb[s % QD][0], q1 = qb[s % QD][1];
        if (s + QD - 1 < NCH) ldg_nc_v8(Qrow + 64 * (s + QD - 1), qb[(s + QD - 1) % QD][0], qb[(s + QD - 1) % QD][1]);
        uint4 p0, p1;
        if constexpr (STAGED) {
          p0 = *reinterpret_cast<const uint4*>(prow + 128 * s);
          p1 = *reinterpret_cast<const uint4*>(prow + 128 * s + 16);
        } else {
          p0 = ldg_nc_v4(prow + 128 * s);
          p1 = ldg_nc_v4(prow + 128 * s + 16);
        }
        const uint32_t qw[8] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
        const uint32_t pw[8] = {p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w};
        uint32_t pq[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) pq[j] = tc::h2_add(pw[j], qw[j]);
        tc::tmem_wait_ld();
        uint32_t v[8], ds2[BWD ? 8 : 1];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const uint32_t x = tc::h2_add(tc::pack_f16(__uint_as_float(acc[2 * j]), __uint_as_float(acc[2 * j + 1])), pq[j]);
          const uint32_t t = tc::h2_tanh(x);
          v[j] = tc::h2_fma(x, t, x);
          if (BWD)  // 2 SiLU'(2x) = (1 + t) + s (1 - t)
            ds2[j] = tc::h2_fma(v[j], tc::h2_fma(t, H2_NEG_ONE, H2_ONE), tc::h2_add(t, H2_ONE));
        }
        tc::tmem_st8(TX + tlane + (uint32_t)(64 * s + 16 * g), v);
        if (s == 0 && it > 0) read_out(it - 1, tile - gridDim.x, valid_prev);  // Y of the previous tile, before G2 overwrites it
        // 2 SiLU'(2a') waits for E3 in this thread's own two chunks of the slab E3 will overwrite with abar: the slab
        // is free once its spill copy has read it (GS / G4 of the previous tile are done: read_out has waited for them)
        if constexpr (BWD) {
          if (it > 0) tc::mbar_wait(bar(B_SPILL_S + s), (uint32_t)((it - 1) & 1));
          store_slab(s, ds2);
        }
        publish_tmem(s);
      }
      };
      if (fast) e1_loop(std::true_type{}); else e1_loop(std::false_type{});
      if (!BWD && lane == 0) mbar_arrive(bar(B_X_FREE));  // X is dead: G1 of the next tile may run
      if (lane == 0) mbar_arrive(bar(B_P_FREE));           // staged P rows may be replaced

      // ---- next tile: row metadata and first Q chunk (forward: in flight while the tensor core
      // finishes G2 and during E2; backward: requested between E2 and E3, when the registers of E2 are free) ----
      int rc_n = -1;
      float w_n = 0.f;
      auto fetch_next = [&]() {
        if (!has_next) return;
        tc::mbar_wait(bar(B_META_FULL + (b ^ 1)), (uint32_t)(((it + 1) >> 1) & 1));
        rc_n = meta[b ^ 1].recv[row];
        w_n = meta[b ^ 1].w[row];
        Qrow = a.Qh + (size_t)(rc_n >= 0 ? meta[b ^ 1].send[row] : 0) * D + 16 * g;
#pragma unroll
        for (int s = 0; s < QD - 1; ++s) ldg_nc_v8(Qrow + 64 * s, qb[s][0], qb[s][1]);
      };
      if (!BWD) fetch_next();

      // ---- E2 ----
      if (!BWD) {
        // forward: phi = SiLU(p) -> slabs (weighted by alpha u_e inside the selector of GS)
        tc::mbar_wait(bar(B_D2_FULL), par);
        tc::fence_after_sync();
#pragma unroll
        for (int s = 0; s < NCH; ++s) {
          if (s == NCH / 2) { tc::mbar_wait(bar(B_D2B_FULL), par); tc::fence_after_sync(); }
          uint32_t acc[16];
          tmem_ld16_nowait(TY + tlane + (uint32_t)(64 * s + 16 * g), acc);
          const uint4 c0 = *reinterpret_cast<const uint4*>(b2h + 128 * s);
          const uint4 c1 = *reinterpret_cast<const uint4*>(b2h + 128 * s + 16);
          const uint32_t bw[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
          tc::tmem_wait_ld();
          uint32_t v[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const uint32_t x = tc::h2_add(tc::pack_f16(__uint_as_float(acc[2 * j]), __uint_as_float(acc[2 * j + 1])), bw[j]);
            v[j] = tc::h2_fma(x, tc::h2_tanh(x), x);
          }
          store_slab(s, v);
          publish(s);
        }
      } else {
        // backward: pbar = alpha u mbar_i SiLU'(p) -> slabs ; ubar_e = alpha <mbar_i, phi_e>
        tc::mbar_wait(bar(B_MB_FULL), par);
        const unsigned char* mrow = gen + SM::mtile + myslot * (D * 2) + 32 * g;
        const __half* mrow_g = a.mbar_h + (size_t)(valid ? rc : 0) * D + 16 * g;
        const uint32_t w2 = tc::pack_f16(w, w);
        float ub = 0.f;
        tc::mbar_wait(bar(B_D2_FULL), par);
        tc::fence_after_sync();
        auto e2_loop = [&](auto staged) {
        constexpr bool STAGED = decltype(staged)::value;
#pragma unroll
        for (int s = 0; s < NCH; ++s) {
          if (s == NCH / 2) { tc::mbar_wait(bar(B_D2B_FULL), par); tc::fence_after_sync(); }
          uint32_t acc[16];
          tmem_ld16_nowait(TY + tlane + (uint32_t)(64 * s + 16 * g), acc);
          const uint4 c0 = *reinterpret_cast<const uint4*>(b2h + 128 * s);
          const uint4 c1 = *reinterpret_cast<const uint4*>(b2h + 128 * s + 16);
          const uint32_t bw[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
          uint32_t mb[8];
          if constexpr (STAGED) {
            const uint4 m0 = *reinterpret_cast<const uint4*>(mrow + 128 * s);
            const uint4 m1 = *reinterpret_cast<const uint4*>(mrow + 128 * s + 16);
            mb[0] = m0.x; mb[1] = m0.y; mb[2] = m0.z; mb[3] = m0.w; mb[4] = m1.x; mb[5] = m1.y; mb[6] = m1.z; mb[7] = m1.w;
          } else {
            const uint4 m0 = ldg_nc_v4(mrow_g + 64 * s), m1 = ldg_nc_v4(mrow_g + 64 * s + 8);
            mb[0] = m0.x; mb[1] = m0.y; mb[2] = m0.z; mb[3] = m0.w; mb[4] = m1.x; mb[5] = m1.y; mb[6] = m1.z; mb[7] = m1.w;
          }
          tc::tmem_wait_ld();
          uint32_t v[8];
          uint32_t ubp = 0u;
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const uint32_t x = tc::h2_add(tc::pack_f16(__uint_as_float(acc[2 * j]), __uint_as_float(acc[2 * j + 1])), bw[j]);
            const uint32_t t = tc::h2_tanh(x);
            const uint32_t phi = tc::h2_fma(x, t, x);
            // SiLU'(p) = sigma + phi (1 - sigma), sigma = (1 + t)/2
            const uint32_t dphi = tc::h2_fma(phi, tc::h2_fma(t, H2_NEG_HALF, H2_HALF), tc::h2_fma(t, H2_HALF, H2_HALF));
            ubp = tc::h2_fma(mb[j], phi, ubp);
            v[j] = tc::h2_mul(tc::h2_mul(mb[j], w2), dphi);
          }
          ub += tc::h2_lo(ubp) + tc::h2_hi(ubp);
          tc::tmem_st8(TY + tlane + (uint32_t)(64 * s + 16 * g), v);
          publish_tmem(s);
        }
        };
        if (fast) e2_loop(std::true_type{}); else e2_loop(std::false_type{});
        if (lane == 0) mbar_arrive(bar(B_MB_FREE));
        ubar_s[g * TE + row] = ub;
        fetch_next();

        // ---- E3: abar = X * 2 SiLU'(2a') -> slabs ----
        tc::mbar_wait(bar(B_D3_FULL), par);
        tc::fence_after_sync();
        uint32_t accb[2][16];  // the accumulator columns of slab s + 1 are in flight while slab s is processed
        tmem_ld16_nowait(TX + tlane + (uint32_t)(16 * g), accb[0]);
#pragma unroll
        for (int s = 0; s < NCH; ++s) {
          const uint4 d0 = *reinterpret_cast<const uint4*>(ring + s * SLOT_BYTES + so0);
          const uint4 d1 = *reinterpret_cast<const uint4*>(ring + s * SLOT_BYTES + so1);
          const uint32_t ds2[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
          tc::tmem_wait_ld();
          if (s + 1 < NCH) {
            if (s + 1 == NCH / 2) { tc::mbar_wait(bar(B_D3B_FULL), par); tc::fence_after_sync(); }
            tmem_ld16_nowait(TX + tlane + (uint32_t)(64 * (s + 1) + 16 * g), accb[(s + 1) & 1]);
          }
          const uint32_t (&acc)[16] = accb[s & 1];
          uint32_t v[8];
#pragma unroll
          for (int j = 0; j < 8; ++j)
            v[j] = tc::h2_mul(tc::pack_f16(__uint_as_float(acc[2 * j]), __uint_as_float(acc[2 * j + 1])), ds2[j]);
          store_slab(s, v);
          publish(s);
        }
        if (lane == 0) mbar_arrive(bar(B_X_FREE));
      }

      valid_prev = valid;
      rc = rc_n;
      w = w_n;
    }
    if (it > 0) read_out(it - 1, (int64_t)blockIdx.x + (int64_t)(it - 1) * gridDim.x, valid_prev);
  }

  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<SM::tmem_cols>(tmem);
}

// out[i] = tail[t] + head[t+1] + ... for the segment that starts in tile t and continues beyond it.
// D/4 threads per tile (one float4 of channels each), 1024/D tiles per 256-thread block.
__global__ void __launch_bounds__(256) k_segment_fixup_tc(int64_t E, const int32_t* __restrict__ E_dyn, int D, int64_t n_tiles,
                                                          const int32_t* __restrict__ rowptr,
                                                          const int32_t* __restrict__ recv, const float* __restrict__ head,
                                                          const float* __restrict__ tail, float* __restrict__ out) {
  if (E_dyn) { E = *E_dyn; n_tiles = (E + TE - 1) / TE; }
  const int tpt = D >> 2;  // threads per tile
  const int64_t t = (int64_t)blockIdx.x * (blockDim.x / tpt) + threadIdx.x / tpt;
  const int c = (threadIdx.x % tpt) * 4;
  if (t >= n_tiles) return;
  const int64_t e0 = t * TE, e1 = e0 + TE;
  if (e1 >= E) return;
  const int i = recv[e1 - 1];
  const int64_t s0 = rowptr[i], s1 = rowptr[i + 1];
  if (!(s1 > e1 && s0 >= e0)) return;
  float4 sum = *reinterpret_cast<const float4*>(tail + (size_t)t * D + c);
  for (int64_t t2 = t + 1; t2 * TE < s1; ++t2) {
    const float4 h = *reinterpret_cast<const float4*>(head + (size_t)t2 * D + c);
    sum.x += h.x; sum.y += h.y; sum.z += h.z; sum.w += h.w;
  }
  *reinterpret_cast<float4*>(out + (size_t)i * D + c) = sum;
}

// Qbar_j = sum_{e in in(j)} abar[rev[e]]; abar is the row-major f16 spill [edge][channel] written by the tensor-map stores
template <int D>
__global__ void __launch_bounds__(256) k_gather_rev_tc(int64_t n, int64_t E_act, const int32_t* __restrict__ E_act_dyn,
                                                       const int32_t* __restrict__ rowptr,
                                                       const int32_t* __restrict__ rev, const __half* __restrict__ abar,
                                                       mlip_nodeop* __restrict__ Qbar) {
  if (E_act_dyn) E_act = *E_act_dyn;
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
    if (re >= E_act) continue;  // reverse edge outside this layer's active set: its adjoint is zero and was not written
    const uint4 v = *reinterpret_cast<const uint4*>(base + (size_t)re * (D * 2) + ch * 16);
    const float2 f0 = __half22float2(*reinterpret_cast<const __half2*>(&v.x));
    const float2 f1 = __half22float2(*reinterpret_cast<const __half2*>(&v.y));
    const float2 f2 = __half22float2(*reinterpret_cast<const __half2*>(&v.z));
    const float2 f3 = __half22float2(*reinterpret_cast<const __half2*>(&v.w));
    acc[0] += f0.x; acc[1] += f0.y; acc[2] += f1.x; acc[3] += f1.y;
    acc[4] += f2.x; acc[5] += f2.y; acc[6] += f3.x; acc[7] += f3.y;
  }
  if (NSUB > 1) {
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], 16);
  }
  if (sub == 0) {
    // Qbar is only ever read as a bf16 GEMM operand: stored as the value the operand producer would round it to
    *reinterpret_cast<uint4*>(Qbar + (size_t)j * D + ch * 8) =
        make_uint4(tc::pack_op(acc[0], acc[1]), tc::pack_op(acc[2], acc[3]), tc::pack_op(acc[4], acc[5]), tc::pack_op(acc[6], acc[7]));
  }
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
encode_tiled_fn get_encode_tiled() {
  static encode_tiled_fn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = (encode_tiled_fn)p;
  }
  return fn;
}
// row-major f16 spill [rows][d], stored in boxes of 64 channels x 128 edges out of SWIZZLE_128B slabs
int make_spill_map(mlip_ctx* ctx, __half* abar, int64_t rows, int d, CUtensorMap* map) {
  memset(map, 0, sizeof(*map));
  if (!abar || rows <= 0) return MLIP_OK;
  encode_tiled_fn enc = get_encode_tiled();
  if (!enc) { ctx->set_error("cuTensorMapEncodeTiled not available"); return MLIP_ERR_CUDA; }
  const cuuint64_t gdim[2] = {(cuuint64_t)d, (cuuint64_t)rows};
  const cuuint64_t gstride[1] = {(cuuint64_t)d * 2};
  const cuuint32_t box[2] = {64, (cuuint32_t)TE};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, abar, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { ctx->set_error("cuTensorMapEncodeTiled failed"); return MLIP_ERR_CUDA; }
  return MLIP_OK;
}

template <int D, bool BWD>
int launch_edge_dir(mlip_ctx* ctx, const EdgeArgs& a) {
  const int64_t tiles = (a.E + TE - 1) / TE;
  if (tiles == 0) return MLIP_OK;
  CUtensorMap spill_map;
  MLIP_TRY(make_spill_map(ctx, (BWD && a.node_adjoint) ? a.abar_h : nullptr, tiles * TE, D, &spill_map));
  const size_t smem = ES<D, BWD>::bytes;
  const unsigned grid = (unsigned)(tiles < ctx->num_sms ? tiles : ctx->num_sms);
  MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_edge_tc<D, BWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_edge_tc<D, BWD><<<grid, N_THREADS, smem, ctx->stream>>>(a, tiles, spill_map);
  ctx->launches++;
  if (!BWD || a.node_adjoint) {
    const int64_t tiles_per_block = 256 / (D / 4);
    k_segment_fixup_tc<<<(unsigned)((tiles + tiles_per_block - 1) / tiles_per_block), 256, 0, ctx->stream>>>(
        a.E, a.E_dyn, D, tiles, a.rowptr, a.recv, a.head, a.tail, BWD ? a.Pbar : a.m);
    ctx->launches++;
  }
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
}  // namespace

int64_t mlip_edge_tc_tiles(int64_t E) { return (E + TE - 1) / TE; }

int mlip_edge_forward_tc(mlip_ctx* ctx, int d, const EdgeArgs& a) {
  if (d == 256) return launch_edge_dir<256, false>(ctx, a);
  if (d == 128) return launch_edge_dir<128, false>(ctx, a);
  ctx->set_error("tensor-core edge kernels need d = 128 or 256");
  return MLIP_ERR_UNSUPPORTED;
}
int mlip_edge_backward_tc(mlip_ctx* ctx, int d, const EdgeArgs& a) {
  if (d == 256) return launch_edge_dir<256, true>(ctx, a);
  if (d == 128) return launch_edge_dir<128, true>(ctx, a);
  ctx->set_error("tensor-core edge kernels need d = 128 or 256");
  return MLIP_ERR_UNSUPPORTED;
}
int mlip_gather_rev_tc(mlip_ctx* ctx, int64_t n, int64_t E_act, const int32_t* E_act_dyn, int d, const int32_t* rowptr,
                       const int32_t* rev, const __half* abar, mlip_nodeop* Qbar) {
  if (n <= 0) return MLIP_OK;
  const unsigned grid = (unsigned)((n * 32 + 255) / 256);
  if (d == 256) k_gather_rev_tc<256><<<grid, 256, 0, ctx->stream>>>(n, E_act, E_act_dyn, rowptr, rev, abar, Qbar);
  else if (d == 128) k_gather_rev_tc<128><<<grid, 256, 0, ctx->stream>>>(n, E_act, E_act_dyn, rowptr, rev, abar, Qbar);
  else { ctx->set_error("tensor-core gather needs d = 128 or 256"); return MLIP_ERR_UNSUPPORTED; }
  ctx->launches++;
  return MLIP_OK;
}
