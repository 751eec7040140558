// Three-body (angle) term of the M3GNet-like variant (BASELINE.json config 5; the paper names the
// model family only, PAPER.md:91,119,131 -- the definition is reading R17 / O7 of DESIGN.md):
//   z_k   = sigma(G h_k + g)                                              16 gates per atom and layer
//   S_e   = sum over in-edges e' = (i <- k) != e of the receiver of e, r_e' < r3, of
//           u3(r_e') [Y_l^0(cos theta_ee') g3_n(r_e')]_{4l+n} * z_k        cos theta = rhat_e . rhat_e'
//   t_e   = u3(r_e) S_e  for r_e < r3, else 0;  enters the first edge linear as W3 t_e (edge_f32.cu)
// and its reverse mode: the adjoint tbar_e = W3^T abar_e (edge_f32.cu) is propagated to rbar (through u3 and g3_n), to a
// per-edge VECTOR gradient gvec_e (through cos theta: d c / d rvec_e = (rhat_e' - c rhat_e) / r_e) and to the gates.
// One warp per receiver; the short in-edges of the row are staged in shared memory and every lane owns one staged edge of an
// ordered pair while it loops over the other. No atomics: every output element has exactly one writer. fp32.
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"

namespace {
constexpr int CAP = 128;         // short in-edges per receiver the kernels take (more: MLIP_ERR_UNSUPPORTED through the status word)
// The triplet kernels are launched twice: rows with at most CAP_SMALL short in-edges (all of them in condensed matter at
// r3 = 4 A: mean 27) by a variant with a small staging area (more resident warps per SM), which appends the other rows to
// a list on the device; a fixed small grid of the CAP-entry variant then walks that list. No host round trip in between.
constexpr int CAP_SMALL = 48;
constexpr float INV_SQRT_4PI = 0.28209479177387814f;

template <bool BWD>
struct Staged {                  // one short in-edge of the receiver, as the OTHER edge of a pair sees it
  float hx, hy, hz, inv_r;       // rhat, 1/r
  float w[16];                   // u3 g3_n z_k of this edge (index 4 l + n): what it contributes as the e' of a pair
  float z[BWD ? 16 : 1];         // backward only: tau = tbar u3 of this edge: what it carries as the e of a pair
};

__device__ __forceinline__ void u3_f(float r, float r3, float& u, float& du) {
  float s, c;
  sincospif(r / r3, &s, &c);
  const bool in = r < r3;
  u = in ? 0.5f * (c + 1.0f) : 0.f;
  du = in ? -(1.5707963267948966f / r3) * s : 0.f;
}
__device__ __forceinline__ void g3_f(float r, float r3, float (&g)[4], float (&dg)[4]) {
  const float delta = r3 * (1.0f / 3.0f), gamma = 0.5f / (delta * delta);
#pragma unroll
  for (int n = 0; n < 4; ++n) {
    const float diff = r - (float)n * delta;
    g[n] = expf(-gamma * diff * diff);
    dg[n] = -2.0f * gamma * diff * g[n];
  }
}
// Y_l^0(c) and d/dc, l = 0..3
__device__ __forceinline__ void ylm(float c, float (&Y)[4], float (&dY)[4]) {
  const float n1 = 1.7320508075688772f * INV_SQRT_4PI, n2 = 2.23606797749979f * INV_SQRT_4PI, n3 = 2.6457513110645907f * INV_SQRT_4PI;
  Y[0] = INV_SQRT_4PI; dY[0] = 0.f;
  Y[1] = n1 * c; dY[1] = n1;
  Y[2] = n2 * (1.5f * c * c - 0.5f); dY[2] = n2 * 3.0f * c;
  Y[3] = n3 * (2.5f * c * c * c - 1.5f * c); dY[3] = n3 * (7.5f * c * c - 1.5f);
}

// z[i, 0..15] = sigma(G h_i + g): one warp per atom
__global__ void __launch_bounds__(256) k_gate(int64_t n, int d, const float* __restrict__ h, const float* __restrict__ G,
                                              const float* __restrict__ g, float* __restrict__ z) {
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= n) return;
  float acc[16];
#pragma unroll
  for (int b = 0; b < 16; ++b) acc[b] = 0.f;
  for (int c = lane; c < d; c += 32) {
    const float x = h[i * d + c];
#pragma unroll
    for (int b = 0; b < 16; ++b) acc[b] = fmaf(G[b * d + c], x, acc[b]);
  }
#pragma unroll
  for (int b = 0; b < 16; ++b)
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) acc[b] += __shfl_xor_sync(0xffffffffu, acc[b], s);
  if (lane < 16) {
    float v = 0.f;
#pragma unroll
    for (int b = 0; b < 16; ++b) if (b == lane) v = acc[b];
    z[i * 16 + lane] = 1.0f / (1.0f + expf(-(v + g[lane])));
  }
}

// number of short in-edges of the row [lo, hi) (warp-uniform)
__device__ __forceinline__ int count_short(int lo, int hi, float r3, const float4* __restrict__ rvec, int lane) {
  int ns = 0;
  for (int b = lo; b < hi; b += 32) {
    const int e = b + lane;
    ns += __popc(__ballot_sync(0xffffffffu, e < hi && rvec[e].w < r3));
  }
  return ns;
}
// Row of this warp: the small-capacity variant takes receiver blockIdx * WARPS + warp and appends rows with more than
// CAP_SMALL short in-edges to long_rows (long_rows[0] = how many, then the receivers); the CAP variant walks that list with a
// grid-stride loop. Returns false when there is nothing (more) to do.
template <int CAP_, int WARPS_>
__device__ __forceinline__ bool next_row(int64_t n, int* __restrict__ long_rows, int lane, int w, int& k, int64_t& i) {
  if (CAP_ == CAP_SMALL) {
    if (k > 0) return false;
    i = (int64_t)blockIdx.x * WARPS_ + w;
    k = 1;
    return i < n;
  }
  const int idx = k * (int)gridDim.x * WARPS_ + (int)blockIdx.x * WARPS_ + w;
  ++k;
  if (idx >= *reinterpret_cast<volatile int*>(long_rows)) return false;
  i = long_rows[1 + idx];
  return true;
}

// Stage the short in-edges of the row [lo, hi) into S[0..min(ns, CAP_)): directions and the 16 products u3 g3_n z_k
template <int CAP_, bool BWD>
__device__ __forceinline__ void stage_row(int lo, int hi, float r3, const float4* __restrict__ rvec,
                                          const int32_t* __restrict__ send, const float* __restrict__ z, Staged<BWD>* S,
                                          int* idx /*[CAP_] edge id of every staged entry*/, int lane) {
  int ns = 0;
  for (int b = lo; b < hi; b += 32) {
    const int e = b + lane;
    float4 rv = make_float4(0.f, 0.f, 0.f, 1e30f);
    if (e < hi) rv = rvec[e];
    const bool ok = e < hi && rv.w < r3;
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    const int slot = ns + __popc(m & ((1u << lane) - 1u));
    if (ok && slot < CAP_) {
      Staged<BWD>& s = S[slot];
      const float inv = rv.w > 0.f ? 1.0f / rv.w : 0.f;
      s.hx = rv.x * inv; s.hy = rv.y * inv; s.hz = rv.z * inv; s.inv_r = inv;
      float u, du, g[4], dg[4];
      u3_f(rv.w, r3, u, du);
      g3_f(rv.w, r3, g, dg);
      const float4* zk = reinterpret_cast<const float4*>(z + (size_t)send[e] * 16);
#pragma unroll
      for (int q4 = 0; q4 < 4; ++q4) {
        const float4 v = zk[q4];
        s.w[4 * q4] = u * g[0] * v.x; s.w[4 * q4 + 1] = u * g[1] * v.y; s.w[4 * q4 + 2] = u * g[2] * v.z; s.w[4 * q4 + 3] = u * g[3] * v.w;
      }
      idx[slot] = e;
    }
    ns += __popc(m);
  }
  __syncwarp();
}

// forward: t[e, 16] for every edge of the receivers [0, n) (zeros for r_e >= r3). Every lane owns one staged (short) edge
// as the e of the pairs (e, p) and loops over the other staged edges p.
template <int CAP_, int WARPS_>
__global__ void __launch_bounds__(WARPS_ * 32) k_triplet_fwd(int64_t n, float r3, const int32_t* __restrict__ rowptr,
                                                             const int32_t* __restrict__ send, const float4* __restrict__ rvec,
                                                             const float* __restrict__ z, float* __restrict__ t,
                                                             int* __restrict__ status, int* __restrict__ long_rows) {
  __shared__ Staged<false> S_all[WARPS_][CAP_];
  __shared__ int idx_all[WARPS_][CAP_];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  Staged<false>* S = S_all[w];
  int* idx = idx_all[w];
  int k = 0;
  int64_t i;
  while (next_row<CAP_, WARPS_>(n, long_rows, lane, w, k, i)) {
  const int lo = rowptr[i], hi = rowptr[i + 1];
  const int ns_all = count_short(lo, hi, r3, rvec, lane);
  if (CAP_ == CAP_SMALL && ns_all > CAP_SMALL) {
    if (lane == 0) long_rows[1 + atomicAdd(long_rows, 1)] = (int)i;
    continue;
  }
  if (ns_all > CAP_ && lane == 0) atomicOr(status, MLIP_DEV_ROW_TOO_LONG);
  const int ns = ns_all < CAP_ ? ns_all : CAP_;
  stage_row<CAP_, false>(lo, hi, r3, rvec, send, z, S, idx, lane);
  // edges of the row beyond r3 (and beyond the staging area) carry no angle term
  for (int b = lo; b < hi; b += 32) {
    const int e = b + lane;
    if (e < hi && !(rvec[e].w < r3)) {
      float4* dst = reinterpret_cast<float4*>(t + (size_t)e * 16);
      dst[0] = dst[1] = dst[2] = dst[3] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  for (int p0 = 0; p0 < ns; p0 += 32) {
    const int me = p0 + lane;
    if (me >= ns) continue;
    const int e = idx[me];
    const float hx = S[me].hx, hy = S[me].hy, hz = S[me].hz;
    float acc[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) acc[q] = 0.f;
    for (int p = 0; p < ns; ++p) {
      if (p == me) continue;
      const Staged<false>& s = S[p];
      const float c = fmaf(hx, s.hx, fmaf(hy, s.hy, hz * s.hz));
      float Y[4], dY[4];
      ylm(c, Y, dY);
#pragma unroll
      for (int q = 0; q < 16; ++q) acc[q] = fmaf(Y[q >> 2], s.w[q], acc[q]);
    }
    float u, du;
    u3_f(rvec[e].w, r3, u, du);
    float4* dst = reinterpret_cast<float4*>(t + (size_t)e * 16);
#pragma unroll
    for (int q4 = 0; q4 < 4; ++q4) dst[q4] = make_float4(acc[4 * q4] * u, acc[4 * q4 + 1] * u, acc[4 * q4 + 2] * u, acc[4 * q4 + 3] * u);
  }
  __syncwarp();   // the staging area is reused by the next row of this warp
  }
}

// reverse mode. In: tbar[e,16]. Out: rbar[e] += ..., gvec[e] += ..., zeta[e,16] = adjoint of the gate of the SENDER of e
// collected per edge (summed over the out-edges of an atom by k_gate_bwd through rev[]).
template <int CAP_, int WARPS_>
__global__ void __launch_bounds__(WARPS_ * 32) k_triplet_bwd(int64_t n, float r3, const int32_t* __restrict__ rowptr,
                                                             const int32_t* __restrict__ send, const float4* __restrict__ rvec,
                                                             const float* __restrict__ z, const float* __restrict__ tbar,
                                                             float* __restrict__ rbar, float4* __restrict__ gvec,
                                                             float* __restrict__ zeta, int* __restrict__ long_rows) {
  __shared__ Staged<true> S_all[WARPS_][CAP_];
  __shared__ int idx_all[WARPS_][CAP_];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  Staged<true>* S = S_all[w];
  int* idx = idx_all[w];
  int k = 0;
  int64_t i;
  while (next_row<CAP_, WARPS_>(n, long_rows, lane, w, k, i)) {
  const int lo = rowptr[i], hi = rowptr[i + 1];
  const int ns_all = count_short(lo, hi, r3, rvec, lane);
  if (CAP_ == CAP_SMALL && ns_all > CAP_SMALL) {
    if (lane == 0) long_rows[1 + atomicAdd(long_rows, 1)] = (int)i;
    continue;
  }
  const int ns = ns_all < CAP_ ? ns_all : CAP_;   // a longer row was reported by the forward kernel
  stage_row<CAP_, true>(lo, hi, r3, rvec, send, z, S, idx, lane);
  // every staged entry also carries tau = tbar u3 of its own edge (pass B reads it as the "e" side)
  for (int p = lane; p < ns; p += 32) {
    const int e = idx[p];
    float u, du;
    u3_f(rvec[e].w, r3, u, du);
    const float4* tb = reinterpret_cast<const float4*>(tbar + (size_t)e * 16);
#pragma unroll
    for (int q4 = 0; q4 < 4; ++q4) {
      const float4 v = tb[q4];
      S[p].z[4 * q4] = v.x * u; S[p].z[4 * q4 + 1] = v.y * u; S[p].z[4 * q4 + 2] = v.z * u; S[p].z[4 * q4 + 3] = v.w * u;
    }
  }
  __syncwarp();
  // edges of the row beyond r3 take part in nothing: their zeta is zero
  for (int b = lo; b < hi; b += 32) {
    const int e = b + lane;
    if (e < hi && !(rvec[e].w < r3)) {
      float4* dst = reinterpret_cast<float4*>(zeta + (size_t)e * 16);
      dst[0] = dst[1] = dst[2] = dst[3] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  for (int p0 = 0; p0 < ns; p0 += 32) {
    const int me = p0 + lane;          // this lane's staged edge, in both roles
    if (me >= ns) continue;
    const int e = idx[me];
    const float4 rv = rvec[e];
    const Staged<true>& my = S[me];
    const float hx = my.hx, hy = my.hy, hz = my.hz;
    float u, du, g[4], dg[4];
    u3_f(rv.w, r3, u, du);
    g3_f(rv.w, r3, g, dg);
    float tb[16], zk[16];
    {
      const float4* src = reinterpret_cast<const float4*>(tbar + (size_t)e * 16);
      const float4* zs = reinterpret_cast<const float4*>(z + (size_t)send[e] * 16);
#pragma unroll
      for (int q4 = 0; q4 < 4; ++q4) {
        const float4 v = src[q4], y = zs[q4];
        tb[4 * q4] = v.x; tb[4 * q4 + 1] = v.y; tb[4 * q4 + 2] = v.z; tb[4 * q4 + 3] = v.w;
        zk[4 * q4] = y.x; zk[4 * q4 + 1] = y.y; zk[4 * q4 + 2] = y.z; zk[4 * q4 + 3] = y.w;
      }
    }
    // ---- pass A: this lane's edge is e of the pairs (e, p): through u3(r_e) and through cos theta on the e side ----
    float tS = 0.f, vx = 0.f, vy = 0.f, vz = 0.f, cc = 0.f;
    // ---- pass B: this lane's edge is e' of the pairs (q, e'): through u3(r_e'), g3_n(r_e'), cos theta, the gate ----
    float D[4], Z[16], rb = 0.f, wx = 0.f, wy = 0.f, wz = 0.f, dd = 0.f;
#pragma unroll
    for (int q = 0; q < 4; ++q) D[q] = du * g[q] + u * dg[q];
#pragma unroll
    for (int q = 0; q < 16; ++q) Z[q] = 0.f;
    for (int p = 0; p < ns; ++p) {
      if (p == me) continue;
      const Staged<true>& s = S[p];
      const float c = fmaf(hx, s.hx, fmaf(hy, s.hy, hz * s.hz));
      float Y[4], dY[4];
      ylm(c, Y, dY);
      // A: A'_l = sum_n tbar_e[4l+n] w_p[4l+n]
      float sY = 0.f, sdY = 0.f;
      // B: B_l = sum_n tau_p[4l+n] z_k[4l+n] D_n ; C_l = sum_n tau_p[4l+n] z_k[4l+n] g_n
      float bY = 0.f, bdY = 0.f;
#pragma unroll
      for (int l = 0; l < 4; ++l) {
        float a = 0.f, bl = 0.f, cl = 0.f;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          a = fmaf(tb[4 * l + q], s.w[4 * l + q], a);
          const float tz = s.z[4 * l + q] * zk[4 * l + q];
          bl = fmaf(tz, D[q], bl);
          cl = fmaf(tz, g[q], cl);
          Z[4 * l + q] = fmaf(s.z[4 * l + q], Y[l], Z[4 * l + q]);
        }
        sY = fmaf(Y[l], a, sY); sdY = fmaf(dY[l], a, sdY);
        bY = fmaf(Y[l], bl, bY); bdY = fmaf(dY[l], cl, bdY);
      }
      tS += sY;
      const float cbarA = u * sdY;     // d/dc of the pair (e = mine, e' = p)
      vx = fmaf(cbarA, s.hx, vx); vy = fmaf(cbarA, s.hy, vy); vz = fmaf(cbarA, s.hz, vz); cc = fmaf(cbarA, c, cc);
      rb += bY;
      const float cbarB = u * bdY;     // d/dc of the pair (e = p, e' = mine)
      wx = fmaf(cbarB, s.hx, wx); wy = fmaf(cbarB, s.hy, wy); wz = fmaf(cbarB, s.hz, wz); dd = fmaf(cbarB, c, dd);
    }
    rbar[e] += du * tS + rb;
    const float inv = my.inv_r;
    float4 gv = gvec[e];
    gv.x += inv * ((vx + wx) - (cc + dd) * hx);
    gv.y += inv * ((vy + wy) - (cc + dd) * hy);
    gv.z += inv * ((vz + wz) - (cc + dd) * hz);
    gvec[e] = gv;
    float4* dst = reinterpret_cast<float4*>(zeta + (size_t)e * 16);
#pragma unroll
    for (int q4 = 0; q4 < 4; ++q4)
      dst[q4] = make_float4(Z[4 * q4] * u * g[0], Z[4 * q4 + 1] * u * g[1], Z[4 * q4 + 2] * u * g[2], Z[4 * q4 + 3] * u * g[3]);
  }
  __syncwarp();   // the staging area is reused by the next row of this warp
  }
}

// zbar_k = sum over in-edges e of k with rev[e] < E_act of zeta[rev[e]]; hbar_k += G^T (zbar_k * z_k (1 - z_k))
__global__ void __launch_bounds__(256) k_gate_bwd(int64_t n, int64_t E_act, const int32_t* __restrict__ E_act_dyn, int d,
                                                  const int32_t* __restrict__ rowptr,
                                                  const int32_t* __restrict__ rev, const float* __restrict__ zeta,
                                                  const float* __restrict__ z, const float* __restrict__ G,
                                                  float* __restrict__ hbar) {
  if (E_act_dyn) E_act = *E_act_dyn;
  const int lane = threadIdx.x & 31;
  const int64_t k = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (k >= n) return;
  const int b = lane & 15, sub = lane >> 4;
  float acc = 0.f;
  for (int e = rowptr[k] + sub; e < rowptr[k + 1]; e += 2) {
    const int re = rev[e];
    if (re < E_act) acc += zeta[(size_t)re * 16 + b];
  }
  acc += __shfl_down_sync(0xffffffffu, acc, 16);
  const float zk = z[k * 16 + b];
  const float pre = acc * zk * (1.0f - zk);      // valid in lanes 0..15
  for (int c = lane; c < d; c += 32) {
    float s = 0.f;
#pragma unroll
    for (int q = 0; q < 16; ++q) s = fmaf(__shfl_sync(0xffffffffu, pre, q), G[q * d + c], s);
    hbar[k * d + c] += s;
  }
}
inline unsigned nblk(int64_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }
constexpr unsigned LONG_GRID = 148 * 4;   // blocks of the list-walking CAP variant
}  // namespace

int mlip_gate_forward(mlip_ctx* ctx, int64_t n, int d, const float* h, const float* G, const float* g, float* z) {
  if (n <= 0) return MLIP_OK;
  k_gate<<<nblk(n * 32, 256), 256, 0, ctx->stream>>>(n, d, h, G, g, z);
  ctx->launches++;
  return MLIP_OK;
}
int mlip_triplet_forward(mlip_ctx* ctx, int64_t n_recv, float r3, const int32_t* rowptr, const int32_t* send,
                         const float4* rvec, const float* z, float* t, int* long_rows) {
  if (n_recv <= 0) return MLIP_OK;
  cudaMemsetAsync(long_rows, 0, sizeof(int), ctx->stream);
  k_triplet_fwd<CAP_SMALL, 4><<<nblk(n_recv, 4), 128, 0, ctx->stream>>>(n_recv, r3, rowptr, send, rvec, z, t, ctx->dev_status, long_rows);
  k_triplet_fwd<CAP, 2><<<LONG_GRID, 64, 0, ctx->stream>>>(n_recv, r3, rowptr, send, rvec, z, t, ctx->dev_status, long_rows);
  ctx->launches += 2;
  return MLIP_OK;
}
int mlip_triplet_backward(mlip_ctx* ctx, int64_t n_recv, float r3, const int32_t* rowptr, const int32_t* send,
                          const float4* rvec, const float* z, const float* tbar, float* rbar, float4* gvec, float* zeta,
                          int* long_rows) {
  if (n_recv <= 0) return MLIP_OK;
  cudaMemsetAsync(long_rows, 0, sizeof(int), ctx->stream);
  k_triplet_bwd<CAP_SMALL, 4><<<nblk(n_recv, 4), 128, 0, ctx->stream>>>(n_recv, r3, rowptr, send, rvec, z, tbar, rbar, gvec, zeta, long_rows);
  k_triplet_bwd<CAP, 2><<<LONG_GRID, 64, 0, ctx->stream>>>(n_recv, r3, rowptr, send, rvec, z, tbar, rbar, gvec, zeta, long_rows);
  ctx->launches += 2;
  return MLIP_OK;
}
int mlip_gate_backward(mlip_ctx* ctx, int64_t n_send, int64_t E_act, const int32_t* E_act_dyn, int d, const int32_t* rowptr,
                       const int32_t* rev, const float* zeta, const float* z, const float* G, float* hbar) {
  if (n_send <= 0) return MLIP_OK;
  k_gate_bwd<<<nblk(n_send * 32, 256), 256, 0, ctx->stream>>>(n_send, E_act, E_act_dyn, d, rowptr, rev, zeta, z, G, hbar);
  ctx->launches++;
  return MLIP_OK;
}
