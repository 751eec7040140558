// MLIP_FP32 path of the fused edge kernels (steps A6, A7 and the edge part of A10):
//   forward : gather P_i, Q_j -> a = P_i + Q_j + W1c e_hat -> s = SiLU(a) -> p = W2 s + b2 ->
//             phi = SiLU(p) -> m_i = alpha sum_e u_e phi_e   (receiver-sorted segmented sum)
//   backward: recompute a, s, p; pbar = alpha u mbar_i SiLU'(p); sbar = W2^T pbar;
//             abar = sbar SiLU'(a); spill abar (sender-side adjoint is gathered through rev[]),
//             Pbar_i = sum_e abar_e, ebar = W1c^T abar, rbar_e += d/dr terms (O5).
// One CTA owns a tile of 64 consecutive (receiver-sorted) edges; contractions are fp32 FMA on
// CUDA cores with W2 streamed through shared memory by cp.async. Segments that straddle tiles
// are written as per-tile head/tail partial rows and combined in a fixed order by
// k_segment_fixup: no floating-point atomics anywhere.
#include <stdlib.h>
#include <string.h>
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"

namespace {
constexpr int TE = 64;   // edges per tile
constexpr int KC = 16;   // k rows of W per pipeline stage

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

template <int D>
struct Smem {
  static constexpr int LDS = D + 4;
  static constexpr size_t s_off = 0;
  static constexpr size_t ds_off = s_off + sizeof(float) * TE * LDS;
  static constexpr size_t wt_off(bool bwd) { return bwd ? ds_off + sizeof(float) * TE * LDS : ds_off; }
  static constexpr size_t misc_off(bool bwd) { return wt_off(bwd) + sizeof(float) * 2 * KC * D; }
  // misc: ehat[TE][16], u[TE], du[TE], ubar[TE], r[TE], recv[TE], send[TE], t3[TE][16] (three-body variant)
  static constexpr size_t bytes(bool bwd) { return misc_off(bwd) + sizeof(float) * TE * (16 + 4) + sizeof(int) * TE * 2 + sizeof(float) * TE * 16; }
};

// acc[i][4j+q] += sum_k S[ty*4+i][k] * Wg[k][tx*4 + 64j + q], Wg is [D][D] row-major in global
template <int D>
__device__ __forceinline__ void tile_gemm(const float* __restrict__ S, const float* __restrict__ Wg, float* Wt,
                                          float (&acc)[4][D / 16], int tid, int tx, int ty) {
  constexpr int LDS = D + 4;
  constexpr int V = D / 64;  // float4 per thread per stage, and float4 column groups per thread
  auto load = [&](int c, int buf) {
#pragma unroll
    for (int q = 0; q < V; ++q) {
      const int idx = tid + 256 * q;
      const int kk = idx / (D / 4), c4 = idx % (D / 4);
      cp_async16(Wt + ((size_t)buf * KC + kk) * D + c4 * 4, Wg + (size_t)(c * KC + kk) * D + c4 * 4);
    }
    cp_async_commit();
  };
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < D / 16; ++j) acc[i][j] = 0.f;
  load(0, 0);
  for (int c = 0; c < D / KC; ++c) {
    if (c + 1 < D / KC) { load(c + 1, (c + 1) & 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
    __syncthreads();
    const float* W = Wt + (size_t)(c & 1) * KC * D;
#pragma unroll
    for (int k4 = 0; k4 < KC; k4 += 4) {
      float4 s[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) s[i] = *reinterpret_cast<const float4*>(S + (ty * 4 + i) * LDS + c * KC + k4);
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
#pragma unroll
        for (int j = 0; j < V; ++j) {
          const float4 w = *reinterpret_cast<const float4*>(W + (k4 + kk) * D + tx * 4 + 64 * j);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float sv = kk == 0 ? s[i].x : kk == 1 ? s[i].y : kk == 2 ? s[i].z : s[i].w;
            acc[i][4 * j + 0] = fmaf(sv, w.x, acc[i][4 * j + 0]);
            acc[i][4 * j + 1] = fmaf(sv, w.y, acc[i][4 * j + 1]);
            acc[i][4 * j + 2] = fmaf(sv, w.z, acc[i][4 * j + 2]);
            acc[i][4 * j + 3] = fmaf(sv, w.w, acc[i][4 * j + 3]);
          }
        }
      }
    }
    __syncthreads();
  }
}

// Column sums of X[TE][D] over runs of equal receiver; complete segments go to out[recv],
// segments continuing from an earlier tile to head[tile], segments continuing into a later tile
// to tail[tile].
template <int D>
__device__ __forceinline__ void segmented_store(const float* __restrict__ X, const int* __restrict__ recv_s,
                                                const int32_t* __restrict__ rowptr, int64_t e0, int64_t tile,
                                                float* __restrict__ out, float* __restrict__ head,
                                                float* __restrict__ tail, int tid) {
  constexpr int LDS = D + 4;
  if (tid >= D) return;
  int cur = recv_s[0];
  float sum = 0.f;
  for (int e = 0; e <= TE; ++e) {
    const int r = e < TE ? recv_s[e] : -2;
    if (r != cur) {
      if (cur >= 0) {
        const int64_t s0 = rowptr[cur], s1 = rowptr[cur + 1];
        if (s0 >= e0 && s1 <= e0 + TE) out[(size_t)cur * D + tid] = sum;
        else if (s0 < e0) head[(size_t)tile * D + tid] = sum;
        else tail[(size_t)tile * D + tid] = sum;
      }
      cur = r;
      sum = 0.f;
    }
    if (e < TE && r >= 0) sum += X[e * LDS + tid];
  }
}

template <int D, bool BWD>
__global__ void __launch_bounds__(256, (D <= 128 ? (BWD ? 2 : 3) : 1)) k_edge_f32(EdgeArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using SM = Smem<D>;
  constexpr int LDS = SM::LDS;
  float* S = reinterpret_cast<float*>(smem_raw + SM::s_off);
  float* dS = reinterpret_cast<float*>(smem_raw + SM::ds_off);
  float* Wt = reinterpret_cast<float*>(smem_raw + SM::wt_off(BWD));
  float* ehat = reinterpret_cast<float*>(smem_raw + SM::misc_off(BWD));
  float* u_s = ehat + TE * 16;
  float* du_s = u_s + TE;
  float* ubar_s = du_s + TE;
  float* r_s = ubar_s + TE;
  int* recv_s = reinterpret_cast<int*>(r_s + TE);
  int* send_s = recv_s + TE;
  float* t3_s = reinterpret_cast<float*>(send_s + TE);

  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int64_t tile = blockIdx.x;
  const int64_t e0 = tile * TE;
  const int64_t n_edges = a.E_dyn ? (int64_t)__ldg(a.E_dyn) : a.E;   // Verlet-skin mode: a.E is only the capacity
  if (e0 >= n_edges) return;

  // ---- tile metadata and edge features (A6) ----
  if (tid < TE) {
    const int64_t e = e0 + tid;
    int rc = -1, sd = 0;
    float r = 0.f, u = 0.f, du = 0.f;
    if (e < n_edges) {
      rc = a.recv[e]; sd = a.send[e]; r = a.rvec[e].w;
      envelope_f(r, a.r_cut, u, du);
    }
    recv_s[tid] = rc; send_s[tid] = sd; u_s[tid] = u; du_s[tid] = du; r_s[tid] = r; ubar_s[tid] = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      float g = 0.f, dg;
      if (e < n_edges && k < a.n_rbf) rbf_f(r, a.r_cut, a.n_rbf, k, g, dg);
      ehat[tid * 16 + k] = u * g;
    }
  }
  if (a.t3) {  // three-body variant: the 16 angle terms of every edge of the tile
    for (int idx = tid; idx < TE * 4; idx += 256) {
      const int64_t e = e0 + (idx >> 2);
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (e < n_edges) v = *reinterpret_cast<const float4*>(a.t3 + (size_t)e * 16 + (idx & 3) * 4);
      *reinterpret_cast<float4*>(t3_s + idx * 4) = v;
    }
  }
  __syncthreads();

  // ---- a = P_i + Q_j + W1c e_hat ; s = SiLU(a) ----
  {
    const int col = tid % D, grp = tid / D;
    constexpr int G = 256 / D;
    float w1c[16];
#pragma unroll
    for (int k4 = 0; k4 < 4; ++k4) {
      const float4 w = *reinterpret_cast<const float4*>(a.W1c + (size_t)col * 16 + k4 * 4);
      w1c[4 * k4] = w.x; w1c[4 * k4 + 1] = w.y; w1c[4 * k4 + 2] = w.z; w1c[4 * k4 + 3] = w.w;
    }
    float w3[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) w3[k] = 0.f;
    if (a.t3) {
#pragma unroll
      for (int k4 = 0; k4 < 4; ++k4) {
        const float4 w = *reinterpret_cast<const float4*>(a.W3 + (size_t)col * 16 + k4 * 4);
        w3[4 * k4] = w.x; w3[4 * k4 + 1] = w.y; w3[4 * k4 + 2] = w.z; w3[4 * k4 + 3] = w.w;
      }
    }
    for (int e = grp; e < TE; e += G) {
      const int rc = recv_s[e];
      float s = 0.f, ds = 0.f;
      if (rc >= 0) {
        float v = a.P[(size_t)rc * a.ldp + col] + a.Q[(size_t)send_s[e] * a.ldq + col];
#pragma unroll
        for (int k = 0; k < 16; ++k) v = fmaf(w1c[k], ehat[e * 16 + k], v);
        if (a.t3) {
#pragma unroll
          for (int k = 0; k < 16; ++k) v = fmaf(w3[k], t3_s[e * 16 + k], v);
        }
        silu_both_f(v, s, ds);
      }
      S[e * LDS + col] = s;
      if (BWD) dS[e * LDS + col] = ds;
    }
  }
  __syncthreads();

  // ---- p = W2 s + b2 ----
  float acc[4][D / 16];
  tile_gemm<D>(S, a.W2T, Wt, acc, tid, tx, ty);  // ends with __syncthreads: S may be overwritten

  if (!BWD) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int row = ty * 4 + i;
      const float scale = a.alpha * u_s[row];
#pragma unroll
      for (int j = 0; j < D / 64; ++j) {
        const int c = tx * 4 + 64 * j;
        const float4 b = *reinterpret_cast<const float4*>(a.b2 + c);
        float4 o;
        o.x = scale * silu_f(acc[i][4 * j + 0] + b.x);
        o.y = scale * silu_f(acc[i][4 * j + 1] + b.y);
        o.z = scale * silu_f(acc[i][4 * j + 2] + b.z);
        o.w = scale * silu_f(acc[i][4 * j + 3] + b.w);
        *reinterpret_cast<float4*>(S + row * LDS + c) = o;
      }
    }
    __syncthreads();
    segmented_store<D>(S, recv_s, a.rowptr, e0, tile, a.m, a.head, a.tail, tid);
    return;
  }

  // ---- backward: pbar = alpha u mbar_i SiLU'(p), ubar_e = alpha <mbar_i, phi_e> ----
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int row = ty * 4 + i;
    const int rc = recv_s[row];
    const float au = a.alpha * u_s[row];
    float up = 0.f;
#pragma unroll
    for (int j = 0; j < D / 64; ++j) {
      const int c = tx * 4 + 64 * j;
      const float4 b = *reinterpret_cast<const float4*>(a.b2 + c);
      float4 mb = make_float4(0.f, 0.f, 0.f, 0.f);
      if (rc >= 0) mb = *reinterpret_cast<const float4*>(a.mbar + (size_t)rc * D + c);
      float phi, dphi;
      float4 o;
      silu_both_f(acc[i][4 * j + 0] + b.x, phi, dphi); up = fmaf(mb.x, phi, up); o.x = au * mb.x * dphi;
      silu_both_f(acc[i][4 * j + 1] + b.y, phi, dphi); up = fmaf(mb.y, phi, up); o.y = au * mb.y * dphi;
      silu_both_f(acc[i][4 * j + 2] + b.z, phi, dphi); up = fmaf(mb.z, phi, up); o.z = au * mb.z * dphi;
      silu_both_f(acc[i][4 * j + 3] + b.w, phi, dphi); up = fmaf(mb.w, phi, up); o.w = au * mb.w * dphi;
      *reinterpret_cast<float4*>(S + row * LDS + c) = o;
    }
    // reduce over the 16 column-threads of this row group (lanes tx of a half warp)
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) up += __shfl_xor_sync(0xffffffffu, up, o);
    if (tx == 0) ubar_s[row] = a.alpha * up;
  }
  __syncthreads();

  // ---- sbar = W2^T pbar ; abar = sbar SiLU'(a) ----
  tile_gemm<D>(S, a.W2, Wt, acc, tid, tx, ty);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int row = ty * 4 + i;
    const int64_t e = e0 + row;
#pragma unroll
    for (int j = 0; j < D / 64; ++j) {
      const int c = tx * 4 + 64 * j;
      float4 ds = *reinterpret_cast<const float4*>(dS + row * LDS + c);
      ds.x *= acc[i][4 * j + 0]; ds.y *= acc[i][4 * j + 1]; ds.z *= acc[i][4 * j + 2]; ds.w *= acc[i][4 * j + 3];
      *reinterpret_cast<float4*>(dS + row * LDS + c) = ds;
      if (e < n_edges) *reinterpret_cast<float4*>(a.abar + (size_t)e * D + c) = ds;
    }
  }
  __syncthreads();

  // ---- ebar = W1c^T abar ; rbar_e += ubar u' + sum_k ebar_k (u' g_k + u g'_k) ----
  {
    const int e = tid >> 2, kq = tid & 3;
    float eb[4] = {0.f, 0.f, 0.f, 0.f};
    for (int c = 0; c < D; ++c) {
      const float av = dS[e * LDS + c];
      const float4 w = *reinterpret_cast<const float4*>(a.W1c + (size_t)c * 16 + kq * 4);
      eb[0] = fmaf(av, w.x, eb[0]); eb[1] = fmaf(av, w.y, eb[1]);
      eb[2] = fmaf(av, w.z, eb[2]); eb[3] = fmaf(av, w.w, eb[3]);
    }
    if (a.tbar) {  // three-body variant: tbar_e = W3^T abar_e
      float4 tb = make_float4(0.f, 0.f, 0.f, 0.f);
      for (int c = 0; c < D; ++c) {
        const float av = dS[e * LDS + c];
        const float4 w = *reinterpret_cast<const float4*>(a.W3 + (size_t)c * 16 + kq * 4);
        tb.x = fmaf(av, w.x, tb.x); tb.y = fmaf(av, w.y, tb.y); tb.z = fmaf(av, w.z, tb.z); tb.w = fmaf(av, w.w, tb.w);
      }
      if (e0 + e < n_edges) *reinterpret_cast<float4*>(a.tbar + (size_t)(e0 + e) * 16 + kq * 4) = tb;
    }
    float part = 0.f;
    const float r = r_s[e], u = u_s[e], du = du_s[e];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int k = kq * 4 + q;
      if (k < a.n_rbf) {
        float g, dg;
        rbf_f(r, a.r_cut, a.n_rbf, k, g, dg);
        part = fmaf(eb[q], fmaf(du, g, u * dg), part);
      }
    }
    part += __shfl_xor_sync(0xffffffffu, part, 1);
    part += __shfl_xor_sync(0xffffffffu, part, 2);
    if (kq == 0 && e0 + e < n_edges) a.rbar[e0 + e] += fmaf(ubar_s[e], du, part);
  }
  segmented_store<D>(dS, recv_s, a.rowptr, e0, tile, a.Pbar, a.head, a.tail, tid);
}

// out[i] = tail[t] + head[t+1] + ... for the segment that starts in tile t and continues beyond it
template <int TILE>
__global__ void k_segment_fixup(int64_t E, const int32_t* __restrict__ E_dyn, int D, const int32_t* __restrict__ rowptr,
                                const int32_t* __restrict__ recv, const float* __restrict__ head,
                                const float* __restrict__ tail, float* __restrict__ out) {
  if (E_dyn) E = *E_dyn;
  const int64_t t = blockIdx.x;
  const int64_t e0 = t * TILE, e1 = e0 + TILE;
  if (e1 >= E) return;  // last tile cannot have a continuing segment
  const int i = recv[e1 - 1];
  const int64_t s0 = rowptr[i], s1 = rowptr[i + 1];
  if (!(s1 > e1 && s0 >= e0)) return;
  for (int c = threadIdx.x; c < D; c += blockDim.x) {
    float sum = tail[(size_t)t * D + c];
    for (int64_t t2 = t + 1; t2 * TILE < s1; ++t2) sum += head[(size_t)t2 * D + c];
    out[(size_t)i * D + c] = sum;
  }
}

// Qbar_j = sum_{e in in(j)} abar[rev[e]]  (sender-side adjoint gathered through the reverse index)
__global__ void __launch_bounds__(256) k_gather_rev_f32(int64_t n, int64_t E_act, const int32_t* __restrict__ E_act_dyn, int D,
                                                        const int32_t* __restrict__ rowptr,
                                                        const int32_t* __restrict__ rev, const float* __restrict__ abar,
                                                        float* __restrict__ Qbar) {
  if (E_act_dyn) E_act = *E_act_dyn;
  const int lane = threadIdx.x & 31;
  const int64_t j = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (j >= n) return;
  const int lo = rowptr[j], hi = rowptr[j + 1];
  for (int c0 = 0; c0 < D; c0 += 128) {
    float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
    const int c = c0 + lane * 4;
    if (c < D) {
      for (int e = lo; e < hi; ++e) {
        const int re = rev[e];
        if (re >= E_act) continue;  // not evaluated by this layer: zero adjoint
        const float4 v = *reinterpret_cast<const float4*>(abar + (size_t)re * D + c);
        s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
      }
      *reinterpret_cast<float4*>(Qbar + (size_t)j * D + c) = s;
    }
  }
}

template <int D>
int launch_edge(mlip_ctx* ctx, const EdgeArgs& a, bool bwd) {
  const int64_t tiles = (a.E + TE - 1) / TE;
  if (tiles == 0) return MLIP_OK;
  const size_t smem = Smem<D>::bytes(bwd);
  if (bwd) {
    MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_edge_f32<D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_edge_f32<D, true><<<(unsigned)tiles, 256, smem, ctx->stream>>>(a);
  } else {
    MLIP_CUDA_CHECK(ctx, cudaFuncSetAttribute(k_edge_f32<D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_edge_f32<D, false><<<(unsigned)tiles, 256, smem, ctx->stream>>>(a);
  }
  k_segment_fixup<TE><<<(unsigned)tiles, D < 256 ? D : 256, 0, ctx->stream>>>(a.E, a.E_dyn, D, a.rowptr, a.recv, a.head,
                                                                           a.tail, bwd ? a.Pbar : a.m);
  ctx->launches += 2;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
}  // namespace

int64_t mlip_edge_f32_tiles(int64_t E) { return (E + TE - 1) / TE; }

// MLIP_B200_FP32_EDGE=cuda keeps the CUDA-core kernels of this file at d = 128 too (A/B measurements)
static bool use_x3(int d, const EdgeArgs& a) {
  static const bool cuda_cores = [] { const char* v = getenv("MLIP_B200_FP32_EDGE"); return v && !strcmp(v, "cuda"); }();
  return !cuda_cores && mlip_edge_x3_supported(d, a);
}

int mlip_edge_forward_f32(mlip_ctx* ctx, int d, const EdgeArgs& a) {
  if (use_x3(d, a)) return mlip_edge_forward_x3(ctx, a);
  switch (d) {
    case 64: return launch_edge<64>(ctx, a, false);
    case 128: return launch_edge<128>(ctx, a, false);
    case 256: return launch_edge<256>(ctx, a, false);
  }
  return MLIP_ERR_UNSUPPORTED;
}
int mlip_edge_backward_f32(mlip_ctx* ctx, int d, const EdgeArgs& a) {
  if (use_x3(d, a)) return mlip_edge_backward_x3(ctx, a);
  switch (d) {
    case 64: return launch_edge<64>(ctx, a, true);
    case 128: return launch_edge<128>(ctx, a, true);
    case 256: return launch_edge<256>(ctx, a, true);
  }
  return MLIP_ERR_UNSUPPORTED;
}
int mlip_gather_rev_f32(mlip_ctx* ctx, int64_t n, int64_t E_act, const int32_t* E_act_dyn, int d, const int32_t* rowptr,
                        const int32_t* rev, const float* abar, float* Qbar) {
  if (n <= 0) return MLIP_OK;
  k_gather_rev_f32<<<(unsigned)((n * 32 + 255) / 256), 256, 0, ctx->stream>>>(n, E_act, E_act_dyn, d, rowptr, rev, abar, Qbar);
  ctx->launches++;
  return MLIP_OK;
}
