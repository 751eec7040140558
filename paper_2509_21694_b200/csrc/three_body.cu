// Three-body (angle) term of the M3GNet-like variant (BASELINE.json config 5; the paper names the
// model family only, PAPER.md:91,119,131 -- the definition is reading R17 / O7 of DESIGN.md):
//   z_k   = sigma(G h_k + g)                                              16 gates per atom and layer
//   S_e   = sum over in-edges e' = (i <- k) != e of the receiver of e, r_e' < r3, of
//           u3(r_e') [Y_l^0(cos theta_ee') g3_n(r_e')]_{4l+n} * z_k        cos theta = rhat_e . rhat_e'
//   t_e   = u3(r_e) S_e  for r_e < r3, else 0;  enters the first edge linear as W3 t_e (edge_f32.cu)
// and its reverse mode: the adjoint tbar_e = W3^T abar_e (edge_f32.cu) is propagated to rbar (through u3 and g3_n), to a
// per-edge VECTOR gradient gvec_e (through cos theta: d c / d rvec_e = (rhat_e' - c rhat_e) / r_e) and to the gates.
// One warp per receiver; the short in-edges of the row are staged in shared memory and every lane owns one edge of an
// ordered pair while it loops over the other. No atomics: every output element has exactly one writer. fp32.
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"

namespace {
constexpr int CAP = 128;         // short in-edges per receiver that fit the staging area
constexpr int WARPS = 2;         // receivers per block (2 x 128 staged edges x 144 B = 36 KB of static shared memory)
constexpr float INV_SQRT_4PI = 0.28209479177387814f;

struct Staged {                  // one short in-edge of the receiver, as the OTHER edge of a pair sees it
  float hx, hy, hz, inv_r;       // rhat, 1/r
  float w[16];                   // u3 g3_n z_k of this edge (index 4 l + n): what it contributes as the e' of a pair
  float z[16];                   // backward only: tau = tbar u3 of this edge: what it carries as the e of a pair
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

// Stage the short in-edges of receiver `i` (row [lo, hi)) into S[0..ns): directions and the 16 products u3 g3_n z_k.
// Returns ns (warp-uniform), or -1 when the row holds more than CAP short edges.
__device__ __forceinline__ int stage_row(int lo, int hi, float r3, const float4* __restrict__ rvec,
                                         const int32_t* __restrict__ send, const float* __restrict__ z, Staged* S,
                                         int* idx /*[CAP] edge id of every staged entry*/, int lane) {
  int ns = 0;
  for (int b = lo; b < hi; b += 32) {
    const int e = b + lane;
    float4 rv = make_float4(0.f, 0.f, 0.f, 1e30f);
    if (e < hi) rv = rvec[e];
    const bool ok = e < hi && rv.w < r3;
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    const int slot = ns + __popc(m & ((1u << lane) - 1u));
    if (ok && slot < CAP) {
      Staged& s = S[slot];
      const float inv = rv.w > 0.f ? 1.0f / rv.w : 0.f;
      s.hx = rv.x * inv; s.hy = rv.y * inv; s.hz = rv.z * inv; s.inv_r = inv;
      float u, du, g[4], dg[4];
      u3_f(rv.w, r3, u, du);
      g3_f(rv.w, r3, g, dg);
      const float* zk = z + (size_t)send[e] * 16;
#pragma unroll
      for (int q = 0; q < 16; ++q) s.w[q] = u * g[q & 3] * zk[q];
      idx[slot] = e;
    }
    ns += __popc(m);
  }
  __syncwarp();
  return ns > CAP ? -1 : ns;
}

// forward: t[e, 16] for every edge of the receivers [0, n) (zeros for r_e >= r3)
__global__ void __launch_bounds__(WARPS * 32) k_triplet_fwd(int64_t n, float r3, const int32_t* __restrict__ rowptr,
                                                            const int32_t* __restrict__ send, const float4* __restrict__ rvec,
                                                            const float* __restrict__ z, float* __restrict__ t,
                                                            int* __restrict__ status) {
  __shared__ Staged S_all[WARPS][CAP];
  __shared__ int idx_all[WARPS][CAP];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t i = (int64_t)blockIdx.x * WARPS + w;
  if (i >= n) return;
  Staged* S = S_all[w];
  const int lo = rowptr[i], hi = rowptr[i + 1];
  const int ns = stage_row(lo, hi, r3, rvec, send, z, S, idx_all[w], lane);
  if (ns < 0) { if (lane == 0) atomicOr(status, MLIP_DEV_ROW_TOO_LONG); }
  const int np = ns < 0 ? CAP : ns;
  for (int b = lo; b < hi; b += 32) {
    const int e = b + lane;
    if (e >= hi) continue;
    const float4 rv = rvec[e];
    float acc[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) acc[q] = 0.f;
    if (rv.w < r3) {
      const float inv = rv.w > 0.f ? 1.0f / rv.w : 0.f;
      const float hx = rv.x * inv, hy = rv.y * inv, hz = rv.z * inv;
      for (int p = 0; p < np; ++p) {
        if (idx_all[w][p] == e) continue;
        const Staged& s = S[p];
        const float c = fmaf(hx, s.hx, fmaf(hy, s.hy, hz * s.hz));
        float Y[4], dY[4];
        ylm(c, Y, dY);
#pragma unroll
        for (int q = 0; q < 16; ++q) acc[q] = fmaf(Y[q >> 2], s.w[q], acc[q]);
      }
      float u, du;
      u3_f(rv.w, r3, u, du);
#pragma unroll
      for (int q = 0; q < 16; ++q) acc[q] *= u;
    }
    float4* dst = reinterpret_cast<float4*>(t + (size_t)e * 16);
    dst[0] = make_float4(acc[0], acc[1], acc[2], acc[3]); dst[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
    dst[2] = make_float4(acc[8], acc[9], acc[10], acc[11]); dst[3] = make_float4(acc[12], acc[13], acc[14], acc[15]);
  }
}

// reverse mode. In: tbar[e,16]. Out: rbar[e] += ..., gvec[e] += ..., zeta[e,16] = adjoint of the gate of the SENDER of e
// collected per edge (summed over the out-edges of an atom by k_gate_bwd through rev[]).
__global__ void __launch_bounds__(WARPS * 32) k_triplet_bwd(int64_t n, float r3, const int32_t* __restrict__ rowptr,
                                                            const int32_t* __restrict__ send, const float4* __restrict__ rvec,
                                                            const float* __restrict__ z, const float* __restrict__ tbar,
                                                            float* __restrict__ rbar, float4* __restrict__ gvec,
                                                            float* __restrict__ zeta) {
  __shared__ Staged S_all[WARPS][CAP];
  __shared__ int idx_all[WARPS][CAP];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t i = (int64_t)blockIdx.x * WARPS + w;
  if (i >= n) return;
  Staged* S = S_all[w];
  int* idx = idx_all[w];
  const int lo = rowptr[i], hi = rowptr[i + 1];
  int ns = stage_row(lo, hi, r3, rvec, send, z, S, idx, lane);
  if (ns < 0) ns = CAP;   // reported by the forward kernel
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
    const Staged& my = S[me];
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
      const Staged& s = S[p];
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
}  // namespace

int mlip_gate_forward(mlip_ctx* ctx, int64_t n, int d, const float* h, const float* G, const float* g, float* z) {
  if (n <= 0) return MLIP_OK;
  k_gate<<<nblk(n * 32, 256), 256, 0, ctx->stream>>>(n, d, h, G, g, z);
  ctx->launches++;
  return MLIP_OK;
}
int mlip_triplet_forward(mlip_ctx* ctx, int64_t n_recv, float r3, const int32_t* rowptr, const int32_t* send,
                         const float4* rvec, const float* z, float* t) {
  if (n_recv <= 0) return MLIP_OK;
  k_triplet_fwd<<<nblk(n_recv, WARPS), WARPS * 32, 0, ctx->stream>>>(n_recv, r3, rowptr, send, rvec, z, t, ctx->dev_status);
  ctx->launches++;
  return MLIP_OK;
}
int mlip_triplet_backward(mlip_ctx* ctx, int64_t n_recv, float r3, const int32_t* rowptr, const int32_t* send,
                          const float4* rvec, const float* z, const float* tbar, float* rbar, float4* gvec, float* zeta) {
  if (n_recv <= 0) return MLIP_OK;
  k_triplet_bwd<<<nblk(n_recv, WARPS), WARPS * 32, 0, ctx->stream>>>(n_recv, r3, rowptr, send, rvec, z, tbar, rbar, gvec, zeta);
  ctx->launches++;
  return MLIP_OK;
}
int mlip_gate_backward(mlip_ctx* ctx, int64_t n_send, int64_t E_act, const int32_t* E_act_dyn, int d, const int32_t* rowptr,
                       const int32_t* rev, const float* zeta, const float* z, const float* G, float* hbar) {
  if (n_send <= 0) return MLIP_OK;
  k_gate_bwd<<<nblk(n_send * 32, 256), 256, 0, ctx->stream>>>(n_send, E_act, E_act_dyn, d, rowptr, rev, zeta, z, G, hbar);
  ctx->launches++;
  return MLIP_OK;
}
