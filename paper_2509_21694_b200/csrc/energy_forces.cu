// Host orchestration of one energy-and-force evaluation (steps A6-A12 of SURVEY.md 8(a)):
// embedding, L x (pre-projection, fused edge layer, node update), readout, the hand-written
// reverse pass, force assembly per sub-domain, and the loop over sub-domains
// with root-energy / all-atom-gradient assembly.
#include "common.cuh"
#include "edge.cuh"
#include "mathfn.cuh"
#include "tc_ptx.cuh"

namespace {
inline unsigned nblk(int64_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }

__global__ void k_embed(int64_t n, int d, const int32_t* __restrict__ species, const float* __restrict__ T,
                        float* __restrict__ h, mlip_nodeop* __restrict__ hb /*bf16 copy for the GEMM operands, or null*/) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n * (d / 4)) return;
  const int64_t i = idx / (d / 4);
  const int c = (int)(idx % (d / 4)) * 4;
  const float4 v = *reinterpret_cast<const float4*>(T + (size_t)species[i] * d + c);
  *reinterpret_cast<float4*>(h + i * d + c) = v;
  if (hb) {
    *reinterpret_cast<uint2*>(hb + i * d + c) = make_uint2(tc::pack_op(v.x, v.y), tc::pack_op(v.z, v.w));
  }
}

// E_i = wo . SiLU(o_i) + b_E + E0[z_i];  obar_i = omega_i wo * SiLU'(o_i)   (O4, first line of O5)
__global__ void __launch_bounds__(256) k_readout(int64_t n, int d, const float* __restrict__ o,
                                                 const float* __restrict__ wo, const float* __restrict__ bE,
                                                 const float* __restrict__ E0, const int32_t* __restrict__ species,
                                                 const float* __restrict__ omega, float* __restrict__ E_i,
                                                 float* __restrict__ obar) {
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= n) return;
  const float w = omega ? omega[i] : 1.0f;
  float acc = 0.f;
  for (int c = lane * 4; c < d; c += 128) {
    const float4 x = *reinterpret_cast<const float4*>(o + i * d + c);
    const float4 q = *reinterpret_cast<const float4*>(wo + c);
    float s, ds;
    float4 ob;
    silu_both_f(x.x, s, ds); acc = fmaf(q.x, s, acc); ob.x = w * q.x * ds;
    silu_both_f(x.y, s, ds); acc = fmaf(q.y, s, acc); ob.y = w * q.y * ds;
    silu_both_f(x.z, s, ds); acc = fmaf(q.z, s, acc); ob.z = w * q.z * ds;
    silu_both_f(x.w, s, ds); acc = fmaf(q.w, s, acc); ob.w = w * q.w * ds;
    *reinterpret_cast<float4*>(obar + i * d + c) = ob;
  }
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
  if (lane == 0) E_i[i] = acc + bE[0] + E0[species[i]];
}

// ---- power-of-two scale of the reverse pass (MLIP_BF16 only) -----------------------------------------------------
// The reverse pass is linear in obar = d(sum of root energies)/d o, so obar may be multiplied by any s as long as the
// per-edge adjoints rbar are divided by s when the forces and the virial are assembled. With s = 2^k chosen such that
// max |s obar| lies in [2, 4), the f16 adjoints of the tensor-core edge kernels (mbar, pbar, abar) sit 14 octaves above
// the f16 subnormals and 14 below its maximum whatever the energy scale of the model; a power of two changes no
// mantissa. scale[0] = s, scale[1] = 1/s.
__global__ void __launch_bounds__(256) k_absmax_partial(int64_t n, const float* __restrict__ x, float* __restrict__ partial) {
  __shared__ float sh[256];
  float m = 0.f;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    m = fmaxf(m, fabsf(x[i]));  // fmaxf drops NaN: a NaN in obar reaches the forces and is reported there
  sh[threadIdx.x] = m;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] = fmaxf(sh[threadIdx.x], sh[threadIdx.x + s]);
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void k_pick_scale(int n_partial, const float* __restrict__ partial, float* __restrict__ scale) {
  if (threadIdx.x != 0) return;
  float m = 0.f;
  for (int i = 0; i < n_partial; ++i) m = fmaxf(m, partial[i]);
  float s = 1.0f;
  if (m > 0.f && m < 3.0e38f) {
    int e;
    frexpf(m, &e);            // m = f 2^e, f in [0.5, 1)  ->  m 2^(2-e) in [2, 4)
    int k = 2 - e;
    k = k > 60 ? 60 : (k < -60 ? -60 : k);
    s = ldexpf(1.0f, k);
  }
  scale[0] = s;
  scale[1] = 1.0f / s;
}
__global__ void k_scale_inplace(int64_t n4, float4* __restrict__ x, const float* __restrict__ scale) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n4) return;
  const float s = scale[0];
  float4 v = x[i];
  v.x *= s; v.y *= s; v.z *= s; v.w *= s;
  x[i] = v;
}

// non-finite energy or force -> sticky context status (MLIP_ERR_NUMERIC at the next synchronising call)
__global__ void k_check_finite(int64_t n, const float* __restrict__ F, const double* __restrict__ energy, int* __restrict__ status) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = i < n && !isfinite(F[i]);
  if (i == 0) bad = bad || !isfinite(energy[0]);
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(status, MLIP_DEV_NONFINITE);
}

// deterministic float64 sum of the root-atom energies: per-block partials, then one block
__global__ void __launch_bounds__(256) k_energy_partial(int64_t n, const float* __restrict__ E_i,
                                                        const float* __restrict__ omega, const int32_t* __restrict__ gid,
                                                        double* __restrict__ partial, float* __restrict__ atom_energy) {
  __shared__ double sh[256];
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double v = 0.0;
  if (i < n) {
    const float w = omega ? omega[i] : 1.0f;
    v = (double)w * (double)E_i[i];
    if (atom_energy && w != 0.f) atom_energy[gid ? gid[i] : i] = E_i[i];
  }
  sh[threadIdx.x] = v;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void __launch_bounds__(256) k_energy_final(int64_t n_partial, const double* __restrict__ partial,
                                                      double* __restrict__ energy) {
  __shared__ double sh[256];
  double v = 0.0;
  for (int64_t i = threadIdx.x; i < n_partial; i += 256) v += partial[i];
  sh[threadIdx.x] = v;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) energy[0] += sh[0];
}

// A11: f_k = sum_{e in in(k)} (rbar_e + rbar_rev(e)) rhat_e ; F[gid_k] += f_k
__global__ void __launch_bounds__(256) k_forces(int64_t n, const int32_t* __restrict__ rowptr,
                                                const int32_t* __restrict__ rev, const float4* __restrict__ rvec,
                                                const float* __restrict__ rbar, const int32_t* __restrict__ gid,
                                                const float* __restrict__ scale /*[2] = s, 1/s of the reverse pass, or null*/,
                                                const float4* __restrict__ gvec /*[E] vector part of dE/d rvec_e (three-body), or null*/,
                                                float* __restrict__ F) {
  const int lane = threadIdx.x & 31;
  const int64_t k = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (k >= n) return;
  const float inv_s = scale ? scale[1] : 1.0f;
  float fx = 0.f, fy = 0.f, fz = 0.f;
  for (int e = rowptr[k] + lane; e < rowptr[k + 1]; e += 32) {
    const float4 rv = rvec[e];
    const int re = rev[e];
    const float w = (rbar[e] + rbar[re]) * (rv.w > 0.f ? inv_s / rv.w : 0.f);
    fx = fmaf(w, rv.x, fx); fy = fmaf(w, rv.y, fy); fz = fmaf(w, rv.z, fz);
    if (gvec) {  // d rvec_e / d x_k = +1 for the in-edges of k, -1 for its out-edges (= the reverse edges)
      const float4 a = gvec[e], b = gvec[re];
      fx += a.x - b.x; fy += a.y - b.y; fz += a.z - b.z;
    }
  }
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) {
    fx += __shfl_xor_sync(0xffffffffu, fx, s);
    fy += __shfl_xor_sync(0xffffffffu, fy, s);
    fz += __shfl_xor_sync(0xffffffffu, fz, s);
  }
  if (lane == 0) {
    const int64_t g = gid ? gid[k] : k;
    F[3 * g] += fx; F[3 * g + 1] += fy; F[3 * g + 2] += fz;
  }
}

// Virial of one sub-domain: W_ab += sum_e rbar_e r_a r_b / r over its directed edges (rbar is zero on the
// edges no layer evaluated). float64 per-block partials in a fixed order, then one block: deterministic, no atomics.
__global__ void __launch_bounds__(256) k_virial_partial(int64_t E, const int32_t* __restrict__ E_dyn, const float4* __restrict__ rvec,
                                                        const float* __restrict__ rbar, const float* __restrict__ scale,
                                                        const float4* __restrict__ gvec, double* __restrict__ partial) {
  __shared__ double sh[6][256];
  double w[6] = {0, 0, 0, 0, 0, 0};
  const double inv_s = scale ? (double)scale[1] : 1.0;
  if (E_dyn) E = *E_dyn;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < E; e += (int64_t)gridDim.x * blockDim.x) {
    const float4 rv = rvec[e];
    if (rv.w > 0.f) {
      const double s = inv_s * (double)rbar[e] / (double)rv.w, x = rv.x, y = rv.y, z = rv.z;
      w[0] += s * x * x; w[1] += s * y * y; w[2] += s * z * z;
      w[3] += s * y * z; w[4] += s * x * z; w[5] += s * x * y;
    }
    if (gvec) {  // three-body variant: dE/d rvec_e has gvec_e on top of rbar_e rhat_e (symmetrised; the total is symmetric)
      const float4 gq = gvec[e];
      const double gx = gq.x, gy = gq.y, gz = gq.z, x = rv.x, y = rv.y, z = rv.z;
      w[0] += gx * x; w[1] += gy * y; w[2] += gz * z;
      w[3] += 0.5 * (gy * z + gz * y); w[4] += 0.5 * (gx * z + gz * x); w[5] += 0.5 * (gx * y + gy * x);
    }
  }
#pragma unroll
  for (int k = 0; k < 6; ++k) sh[k][threadIdx.x] = w[k];
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) {
#pragma unroll
      for (int k = 0; k < 6; ++k) sh[k][threadIdx.x] += sh[k][threadIdx.x + s];
    }
    __syncthreads();
  }
  if (threadIdx.x < 6) partial[(size_t)blockIdx.x * 6 + threadIdx.x] = sh[threadIdx.x][0];
}
__global__ void k_virial_final(int n_partial, const double* __restrict__ partial, double* __restrict__ virial) {
  const int k = threadIdx.x;
  if (k >= 6) return;
  double v = 0.0;
  for (int i = 0; i < n_partial; ++i) v += partial[(size_t)i * 6 + k];
  virial[k] += v;
}
// stress[3][3] = W / V from the accumulated (xx, yy, zz, yz, xz, xy)
__global__ void k_stress_out(const double* __restrict__ virial, double inv_volume, double* __restrict__ stress) {
  if (threadIdx.x != 0) return;
  const double xx = virial[0] * inv_volume, yy = virial[1] * inv_volume, zz = virial[2] * inv_volume;
  const double yz = virial[3] * inv_volume, xz = virial[4] * inv_volume, xy = virial[5] * inv_volume;
  stress[0] = xx; stress[1] = xy; stress[2] = xz;
  stress[3] = xy; stress[4] = yy; stress[5] = yz;
  stress[6] = xz; stress[7] = yz; stress[8] = zz;
}

// The tensor-core edge kernels (with their fix-up) write the whole row of every receiver that has at least one edge, so
// only the rows of atoms WITHOUT in-edges have to be cleared -- 4 bytes read per atom instead of 4 d bytes written.
__global__ void __launch_bounds__(256) k_zero_isolated_rows(int64_t n, int d, const int32_t* __restrict__ rowptr,
                                                            float* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= n || rowptr[i + 1] != rowptr[i]) return;
  for (int c = lane * 4; c < d; c += 128) *reinterpret_cast<float4*>(out + i * d + c) = make_float4(0.f, 0.f, 0.f, 0.f);
}

__global__ void k_unpermute(int64_t N, const int32_t* __restrict__ perm, const float* __restrict__ F_int,
                            const float* __restrict__ E_int, float* __restrict__ F_out, float* __restrict__ E_out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  const int64_t a = perm[k];
  F_out[3 * a] = F_int[3 * k]; F_out[3 * a + 1] = F_int[3 * k + 1]; F_out[3 * a + 2] = F_int[3 * k + 2];
  if (E_out) E_out[a] = E_int[k];
}
}  // namespace

int mlip_eval_subgraph(mlip_ctx* ctx, const mlip_model* M, int L, const SubGraph& g, int precision,
                       double* energy_accum, float* F_int, float* Ei_int, double* virial_accum) {
  const int64_t n = g.n, E = g.E;
  if (n == 0) return MLIP_OK;
  const int d = M->h.d;
  const bool bf = precision == MLIP_BF16;
  cudaStream_t st = ctx->stream;
  auto gemm_raw = bf ? mlip_gemm_bf16 : mlip_gemm_f32;
  auto gemm = [&](mlip_ctx* c, const GemmArgs& ga) { ProfScope p(c, MLIP_PROF_NODE_GEMM); return gemm_raw(c, ga); };
  const int64_t tiles = bf ? mlip_edge_tc_tiles(E) : mlip_edge_f32_tiles(E);

  std::vector<void*> ws;
  auto release = [&]() { for (void* p : ws) ctx->free(p); };
#define W_ALLOC(ptr, T, count)                                         \
  do {                                                                 \
    int _s = ctx->alloc(&ptr, (size_t)(count));                        \
    if (_s != MLIP_OK) { release(); return _s; }                       \
    ws.push_back(ptr);                                                 \
  } while (0)
#define W_TRY(x) do { int _s = (x); if (_s != MLIP_OK) { release(); return _s; } } while (0)

  std::vector<float*> h(L + 1), P(L), c(L);
  std::vector<float*> Qf(L, nullptr);
  std::vector<__half*> Ph(L, nullptr), Qh(L, nullptr);
  for (int l = 0; l <= L; ++l) W_ALLOC(h[l], float, n * d);
  for (int l = 0; l < L; ++l) {
    if (bf) {  // layer 0 holds the S-row species tables (section 5b of DESIGN.md), the others one row per atom
      const int64_t rows = l == 0 ? (int64_t)M->h.n_species : n;
      W_ALLOC(Ph[l], __half, rows * d); W_ALLOC(Qh[l], __half, rows * d);
    }
    else { W_ALLOC(P[l], float, n * 2 * d); Qf[l] = P[l] + d; }
    W_ALLOC(c[l], float, n * d);
  }
  float *m = nullptr, *o = nullptr, *hbar = nullptr, *cbar = nullptr, *PQbar = nullptr, *head = nullptr, *tail = nullptr,
        *rbar = nullptr, *E_i = nullptr, *abar = nullptr;
  __half *abar_h = nullptr, *mbar_h = nullptr;
  // tensor-core path: tensors that are only ever read as bf16 GEMM operands are STORED as bf16 -- the value the operand
  // producer would round the fp32 form to, so results do not change while the HBM-bound node GEMMs move fewer bytes:
  // hb = copy of the residual stream h^l (two buffers, alternating), cbar_b, Qbar_b
  mlip_nodeop *hb[2] = {nullptr, nullptr}, *cbar_b = nullptr, *Qbar_b = nullptr;
  double* partial = nullptr;
  float* scale = nullptr;  // [2 + 1184]: s, 1/s of the reverse pass (MLIP_BF16), then the per-block maxima
  if (bf) {
    W_ALLOC(scale, float, 2 + 148 * 8);
    W_ALLOC(hb[0], mlip_nodeop, n * d); W_ALLOC(hb[1], mlip_nodeop, n * d);
    W_ALLOC(cbar_b, mlip_nodeop, n * d); W_ALLOC(Qbar_b, mlip_nodeop, n * d);
  }
  auto from_h = [&](GemmArgs& a, int l) {  // X1 = h^l
    if (bf) a.X1b = hb[l & 1]; else a.X1 = h[l];
    a.ld1 = d; a.K1 = d;
  };
  W_ALLOC(m, float, n * d); W_ALLOC(o, float, n * d); W_ALLOC(hbar, float, n * d); W_ALLOC(cbar, float, n * d);
  W_ALLOC(PQbar, float, n * 2 * d); W_ALLOC(head, float, (tiles + 1) * d); W_ALLOC(tail, float, (tiles + 1) * d);
  W_ALLOC(rbar, float, E + 1); W_ALLOC(E_i, float, n);
  if (L > 0) { if (bf) { W_ALLOC(abar_h, __half, tiles * 128 * d); W_ALLOC(mbar_h, __half, n * d); } else W_ALLOC(abar, float, E * d); }  // bf16 spill: whole 128-edge tile images
  const int64_t n_part = (n + 255) / 256;
  W_ALLOC(partial, double, n_part);
  // three-body variant (fp32 path): gates per layer, angle terms / their adjoints per edge, vector part of dE/d rvec
  const bool tb = (M->h.flags & MLIP_FLAG_THREE_BODY) != 0 && L > 0;
  const float r3 = M->h.r_cut3;
  std::vector<float*> zg(L, nullptr);
  std::vector<float*> t3(L, nullptr);   // angle terms t_e of every layer, kept for the reverse pass (64 B per edge-layer)
  float* tbar3 = nullptr;
  int* long_rows = nullptr;   // scratch list of the triplet kernels
  float4* gvec = nullptr;
  if (tb) {
    for (int l = 0; l < L; ++l) W_ALLOC(zg[l], float, n * 16);
    for (int l = 0; l < L; ++l) W_ALLOC(t3[l], float, (E + 1) * 16);
    W_ALLOC(tbar3, float, (E + 1) * 16); W_ALLOC(long_rows, int, n + 1); W_ALLOC(gvec, float4, E + 1);
    cudaMemsetAsync(gvec, 0, sizeof(float4) * (E + 1), st);
  }
  float* mbar = m;           // m is dead after the forward pass
  float* Pbar = PQbar;
  float* Qbar = PQbar + n * d;  // stored as two dense [n,d] blocks

  {
    ProfScope p(ctx, MLIP_PROF_READOUT_FORCES);
    k_embed<<<nblk(n * (d / 4), 256), 256, 0, st>>>(n, d, g.species, M->T, h[0], hb[0]);
    ctx->launches++;
  }

  EdgeArgs ea;
  ea.E = E; ea.n = n; ea.rowptr = g.rowptr; ea.recv = g.recv; ea.send = g.send; ea.rev = g.rev; ea.rvec = g.rvec;
  ea.r_cut = M->h.r_cut; ea.alpha = M->h.agg_scale; ea.n_rbf = M->h.n_rbf; ea.head = head; ea.tail = tail;

  auto set_layer = [&](int l) {
    const LayerWeights& W = M->layers[l];
    ea.P = P[l]; ea.ldp = 2 * d; ea.Q = Qf[l]; ea.ldq = 2 * d; ea.Ph = Ph[l]; ea.Qh = Qh[l];
    ea.row_index = (bf && l == 0) ? g.species : nullptr;  // P^0, Q^0 are per-species tables (below)
    ea.W1c = W.W1c; ea.W2T = W.W2T; ea.W2 = W.W2; ea.b2 = W.b2;
    ea.W2img = W.W2img; ea.W1cimg = W.W1cimg; ea.W2x3 = W.W2x3; ea.W13x3 = W.W13x3;
  };

  // Active sets (SubGraph depth classes): layer l runs on receivers [0, nr) = classes <= L-1-l, reads senders
  // [0, ns) = classes <= L-l and therefore evaluates the edge prefix [0, Er). Rows beyond nr of h[l+1] are never read.
  const bool act = ctx->active_sets;
  auto n_recv = [&](int l) { return act ? g.atoms_upto(L - 1 - l) : n; };
  auto n_send = [&](int l) { return act ? g.atoms_upto(L - l) : n; };
  auto e_recv = [&](int l) { return act ? g.edges_upto(L - 1 - l) : E; };
  const int64_t n0 = act ? g.atoms_upto(0) : n;  // root atoms (everything when there are no classes)

  for (int l = 0; l < L; ++l) {
    const LayerWeights& W = M->layers[l];
    const int64_t nr = n_recv(l), ns = n_send(l);
    GemmArgs a;
    if (bf && l == 0) {
      // h^0_i = T[z_i]: the pre-projections of the first layer are S-row tables, P^0 = W1a T + b1, Q^0 = W1b T, indexed
      // by species inside the edge kernels (EdgeArgs::row_index)
      a = GemmArgs(); a.X1 = M->T; a.ld1 = d; a.K1 = d; a.B = W.W1a_bf; a.bias = W.b1h; a.Yh = Ph[l]; a.ldy = d; a.n = M->h.n_species; a.N = d;
      W_TRY(gemm(ctx, a));
      a = GemmArgs(); a.X1 = M->T; a.ld1 = d; a.K1 = d; a.B = W.W1b_bf; a.Yh = Qh[l]; a.ldy = d; a.n = M->h.n_species; a.N = d;
      W_TRY(gemm(ctx, a));
    } else if (bf) {
      a = GemmArgs(); from_h(a, l); a.B = W.W1a_bf; a.bias = W.b1h; a.Yh = Ph[l]; a.ldy = d; a.n = nr; a.N = d;
      W_TRY(gemm(ctx, a));
      a = GemmArgs(); from_h(a, l); a.B = W.W1b_bf; a.Yh = Qh[l]; a.ldy = d; a.n = ns; a.N = d;
      W_TRY(gemm(ctx, a));
    } else {
      a = GemmArgs(); a.X1 = h[l]; a.ld1 = d; a.K1 = d; a.B = W.W1ab; a.bias = W.b1pad; a.Y = P[l]; a.ldy = 2 * d; a.n = ns; a.N = 2 * d;
      W_TRY(gemm(ctx, a));
    }
    if (bf) {
      if (nr > 0) { k_zero_isolated_rows<<<nblk(nr * 32, 256), 256, 0, st>>>(nr, d, g.rowptr, m); ctx->launches++; }
    } else {
      cudaMemsetAsync(m, 0, sizeof(float) * nr * d, st);
    }
    set_layer(l);
    ea.m = m; ea.E = e_recv(l); ea.n = nr; ea.E_dyn = g.dyn ? g.rowptr + nr : nullptr;
    if (tb) {
      ProfScope p(ctx, MLIP_PROF_THREE_BODY);
      W_TRY(mlip_gate_forward(ctx, ns, d, h[l], W.G3, W.g3, zg[l]));
      W_TRY(mlip_triplet_forward(ctx, nr, r3, g.rowptr, g.send, g.rvec, zg[l], t3[l], long_rows));
      ea.t3 = t3[l]; ea.W3 = W.W3;
    }
    {
      ProfScope p(ctx, MLIP_PROF_EDGE_FWD);
      W_TRY(bf ? mlip_edge_forward_tc(ctx, d, ea) : mlip_edge_forward_f32(ctx, d, ea));
    }
    a = GemmArgs(); from_h(a, l); a.X2 = m; a.ld2 = d; a.K2 = d;
    a.B = bf ? (const void*)W.V1_bf : (const void*)W.V1; a.bias = W.c1; a.Y = c[l]; a.ldy = d; a.n = nr; a.N = d;
    W_TRY(gemm(ctx, a));
    a = GemmArgs(); a.X1 = c[l]; a.ld1 = d; a.K1 = d; a.act_in = 1;
    a.B = bf ? (const void*)W.V2_bf : (const void*)W.V2; a.bias = W.c2; a.residual = h[l]; a.ldr = d;
    a.Y = h[l + 1]; a.Ybf = bf ? hb[(l + 1) & 1] : nullptr; a.ldy = d; a.n = nr; a.N = d;
    W_TRY(gemm(ctx, a));
  }
  {
    GemmArgs a;
    from_h(a, L); a.B = bf ? (const void*)M->Wo_bf : (const void*)M->Wo; a.bias = M->bo;
    a.Y = o; a.ldy = d; a.n = n0; a.N = d;
    W_TRY(gemm(ctx, a));
  }
  float* obar = cbar;
  {
    ProfScope p(ctx, MLIP_PROF_READOUT_FORCES);
    k_readout<<<nblk(n0 * 32, 256), 256, 0, st>>>(n0, d, o, M->wo, M->bE, M->E0, g.species, g.omega, E_i, obar);
    k_energy_partial<<<(unsigned)((n0 + 255) / 256), 256, 0, st>>>(n0, E_i, g.omega, g.gid, partial, Ei_int);
    k_energy_final<<<1, 256, 0, st>>>((n0 + 255) / 256, partial, energy_accum);
    ctx->launches += 3;
    if (bf && n0 > 0 && L > 0) {
      const int nb = (int)(n0 * d / 4 < 148 * 8 * 256 ? (n0 * d / 4 + 255) / 256 : 148 * 8);
      k_absmax_partial<<<nb, 256, 0, st>>>(n0 * d, obar, scale + 2);
      k_pick_scale<<<1, 32, 0, st>>>(nb, scale + 2, scale);
      k_scale_inplace<<<nblk(n0 * d / 4, 256), 256, 0, st>>>(n0 * d / 4, reinterpret_cast<float4*>(obar), scale);
      ctx->launches += 3;
    }
  }
  const float* rscale = (bf && n0 > 0 && L > 0) ? scale : nullptr;
  {
    GemmArgs a;
    a.X1 = obar; a.ld1 = d; a.K1 = d; a.B = bf ? (const void*)M->WoT_bf : (const void*)M->WoT;
    a.Y = hbar; a.ldy = d; a.n = n0; a.N = d;
    W_TRY(gemm(ctx, a));
  }
  // the adjoint of h^{l+1} is non-zero on the receivers of layer l only; the rows the sender-side GEMM of layer l adds
  // ([nr, ns)) must start from zero
  if (n > n0) cudaMemsetAsync(hbar + n0 * d, 0, sizeof(float) * (n - n0) * d, st);
  cudaMemsetAsync(rbar, 0, sizeof(float) * (E + 1), st);
  for (int l = L - 1; l >= 0; --l) {
    const LayerWeights& W = M->layers[l];
    const int64_t nr = n_recv(l), ns = n_send(l), Er = e_recv(l);
    GemmArgs a;
    a = GemmArgs(); a.X1 = hbar; a.ld1 = d; a.K1 = d; a.B = bf ? (const void*)W.V2T_bf : (const void*)W.V2T;
    a.mul_dsilu = c[l]; a.ldz = d; a.ldy = d; a.n = nr; a.N = d;
    if (bf) a.Ybf = cbar_b; else a.Y = cbar;
    W_TRY(gemm(ctx, a));
    auto from_cbar = [&](GemmArgs& x) { if (bf) x.X1b = cbar_b; else x.X1 = cbar; x.ld1 = d; x.K1 = d; };
    a = GemmArgs(); from_cbar(a); a.B = bf ? (const void*)W.V1bT_bf : (const void*)W.V1bT;
    if (bf) a.Yh = mbar_h; else a.Y = mbar;
    a.ldy = d; a.n = nr; a.N = d;
    W_TRY(gemm(ctx, a));
    // The adjoint of h^0 (the species embedding) is a weight gradient: forces need only rbar. The first layer therefore
    // skips everything that would only feed it: the h-path GEMM, the abar spill, the Pbar sums, the sender-side gather
    // and the projection GEMM.
    const bool node_adjoint = l > 0;
    if (node_adjoint) {
      a = GemmArgs(); from_cbar(a); a.B = bf ? (const void*)W.V1aT_bf : (const void*)W.V1aT;
      a.residual = hbar; a.ldr = d; a.Y = hbar; a.ldy = d; a.n = nr; a.N = d;
      W_TRY(gemm(ctx, a));
    }
    // (the fp32 edge kernel always accumulates its Pbar sums, so its buffer is cleared for the first layer too)
    if (!bf) {
      cudaMemsetAsync(Pbar, 0, sizeof(float) * ns * d, st);
    } else if (node_adjoint) {
      // receivers [0, nr): rows without in-edges; senders that are not receivers of this layer [nr, ns): no Pbar at all
      if (nr > 0) { k_zero_isolated_rows<<<nblk(nr * 32, 256), 256, 0, st>>>(nr, d, g.rowptr, Pbar); ctx->launches++; }
      if (ns > nr) cudaMemsetAsync(Pbar + nr * d, 0, sizeof(float) * (ns - nr) * d, st);
    }
    set_layer(l);
    ea.E = Er; ea.n = nr; ea.node_adjoint = bf ? node_adjoint : true;
    ea.E_dyn = g.dyn ? g.rowptr + nr : nullptr;
    ea.mbar = mbar; ea.mbar_h = mbar_h; ea.abar = abar; ea.abar_h = abar_h; ea.Pbar = Pbar; ea.rbar = rbar;
    if (tb) {  // the angle terms of the forward pass were kept (16 floats per edge-layer; the d-wide activations are recomputed)
      ea.t3 = t3[l]; ea.W3 = W.W3; ea.tbar = tbar3;
    }
    {
      ProfScope p(ctx, MLIP_PROF_EDGE_BWD);
      W_TRY(bf ? mlip_edge_backward_tc(ctx, d, ea) : mlip_edge_backward_f32(ctx, d, ea));
    }
    float* zeta = tb ? t3[l] : nullptr;  // the angle terms are dead after the edge kernel: their buffer takes the per-edge gate adjoints
    if (tb) {
      ProfScope p(ctx, MLIP_PROF_THREE_BODY);
      W_TRY(mlip_triplet_backward(ctx, nr, r3, g.rowptr, g.send, g.rvec, zg[l], tbar3, rbar, gvec, zeta, long_rows));
    }
    if (!node_adjoint) continue;
    {
      ProfScope p(ctx, MLIP_PROF_GATHER_REV);
      // Qbar_j over the senders of this layer, summing only the reverse edges that were evaluated (rev[e] < Er)
      W_TRY(bf ? mlip_gather_rev_tc(ctx, ns, Er, ea.E_dyn, d, g.rowptr, g.rev, abar_h, Qbar_b)
               : mlip_gather_rev_f32(ctx, ns, Er, ea.E_dyn, d, g.rowptr, g.rev, abar, Qbar));
    }
    a = GemmArgs(); a.X1 = Pbar; a.ld1 = d; a.K1 = d; a.ld2 = d; a.K2 = d;
    if (bf) a.X2b = Qbar_b; else a.X2 = Qbar;
    a.B = bf ? (const void*)W.W1abT_bf : (const void*)W.W1abT; a.residual = hbar; a.ldr = d; a.Y = hbar; a.ldy = d;
    a.n = ns; a.N = d;
    W_TRY(gemm(ctx, a));
    if (tb) {  // adjoint of the gates of the senders (third atoms), through the reverse-edge index like Qbar
      ProfScope p(ctx, MLIP_PROF_THREE_BODY);
      W_TRY(mlip_gate_backward(ctx, ns, Er, ea.E_dyn, d, g.rowptr, g.rev, zeta, zg[l], W.G3, hbar));
    }
  }
  {
    ProfScope p(ctx, MLIP_PROF_READOUT_FORCES);
    k_forces<<<nblk(n * 32, 256), 256, 0, st>>>(n, g.rowptr, g.rev, g.rvec, rbar, g.gid, rscale, gvec, F_int);
    ctx->launches++;
    if (virial_accum && E > 0) {
      const int nb = (int)(E < 148 * 8 * 256 ? (E + 255) / 256 : 148 * 8);
      double* vpart = nullptr;
      W_ALLOC(vpart, double, (size_t)nb * 6);
      k_virial_partial<<<nb, 256, 0, st>>>(E, g.dyn ? g.rowptr + n : nullptr, g.rvec, rbar, rscale, gvec, vpart);
      k_virial_final<<<1, 32, 0, st>>>(nb, vpart, virial_accum);
      ctx->launches += 2;
    }
  }
  release();
#undef W_ALLOC
#undef W_TRY
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}

extern "C" int mlip_energy_forces(mlip_ctx* ctx, const mlip_model* M, int L, const mlip_graph* G, const mlip_part* part,
                                  int precision, double* energy_dev, float* forces_dev, float* atom_energy_dev) {
  return mlip_energy_forces_shard(ctx, M, L, G, part, 0, 1, precision, energy_dev, forces_dev, atom_energy_dev);
}

static int energy_forces_impl(mlip_ctx* ctx, const mlip_model* M, int L, const mlip_graph* G, const mlip_part* part,
                              int shard, int n_shards, int precision, double* energy_dev, float* forces_dev,
                              float* atom_energy_dev, double* stress_dev);

extern "C" int mlip_energy_forces_shard(mlip_ctx* ctx, const mlip_model* M, int L, const mlip_graph* G,
                                        const mlip_part* part, int shard, int n_shards, int precision,
                                        double* energy_dev, float* forces_dev, float* atom_energy_dev) {
  return energy_forces_impl(ctx, M, L, G, part, shard, n_shards, precision, energy_dev, forces_dev, atom_energy_dev, nullptr);
}

extern "C" int mlip_energy_forces_stress(mlip_ctx* ctx, const mlip_model* M, int L, const mlip_graph* G,
                                         const mlip_part* part, int shard, int n_shards, int precision,
                                         double* energy_dev, float* forces_dev, float* atom_energy_dev,
                                         double* stress_dev) {
  if (ctx && !stress_dev) { ctx->set_error("mlip_energy_forces_stress: null stress pointer"); return MLIP_ERR_INVALID_ARG; }
  return energy_forces_impl(ctx, M, L, G, part, shard, n_shards, precision, energy_dev, forces_dev, atom_energy_dev, stress_dev);
}

static int energy_forces_impl(mlip_ctx* ctx, const mlip_model* M, int L, const mlip_graph* G, const mlip_part* part,
                              int shard, int n_shards, int precision, double* energy_dev, float* forces_dev,
                              float* atom_energy_dev, double* stress_dev) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (n_shards < 1 || shard < 0 || shard >= n_shards) { ctx->set_error("shard outside [0, n_shards)"); return MLIP_ERR_INVALID_ARG; }
  if (n_shards > 1 && !part) { ctx->set_error("sharded evaluation needs a partition"); return MLIP_ERR_INVALID_ARG; }
  if (part && part->n_shards > 1 && (part->n_shards != n_shards || part->shard != shard)) {
    ctx->set_error("this partition was built for shard " + std::to_string(part->shard) + " of " + std::to_string(part->n_shards) +
                   " (mlip_partition_grid_shard): evaluate it with the same shard and n_shards");
    return MLIP_ERR_INVALID_ARG;
  }
  if (!M || !G || !energy_dev || (G->N > 0 && !forces_dev)) { ctx->set_error("mlip_energy_forces: null argument"); return MLIP_ERR_INVALID_ARG; }
  if (L < 0 || L > M->h.L_max) { ctx->set_error("L outside [0, L_max]"); return MLIP_ERR_UNSUPPORTED; }
  if (precision != MLIP_FP32 && precision != MLIP_BF16) { ctx->set_error("unknown precision"); return MLIP_ERR_INVALID_ARG; }
  if (precision == MLIP_BF16 && !(M->h.d == 256 || M->h.d == 128)) { ctx->set_error("MLIP_BF16 needs d = 128 or 256"); return MLIP_ERR_UNSUPPORTED; }
  if (precision == MLIP_BF16 && (M->h.flags & MLIP_FLAG_THREE_BODY)) {
    ctx->set_error("the three-body variant runs in MLIP_FP32 only (BASELINE.json config 5 is fp32)");
    return MLIP_ERR_UNSUPPORTED;
  }
  if (part && part->N != G->N) { ctx->set_error("partition does not belong to this graph"); return MLIP_ERR_INVALID_ARG; }
  if (part && part->subs.size() > 1 && part->halo < (double)L * (double)M->h.r_cut * (1.0 - 1e-12)) {
    ctx->set_error("halo < L * r_cut: sub-graphs would not keep the K-hop neighbourhood of their root atoms");
    return MLIP_ERR_HALO_TOO_SMALL;
  }
  if (fabs(G->r_cut - (double)M->h.r_cut) > 1e-6 * G->r_cut) { ctx->set_error("graph r_cut differs from model r_cut"); return MLIP_ERR_INVALID_ARG; }
  if (G->N > 0 && (G->species_min < 0 || G->species_max >= M->h.n_species)) {
    ctx->set_error("species outside [0, n_species) of the model");
    return MLIP_ERR_INVALID_ARG;
  }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  const int64_t N = G->N;
  Scratch tmp(ctx);
  float *F_int = nullptr, *E_int = nullptr;
  MLIP_TRY(tmp.get(&F_int, 3 * N));
  MLIP_TRY(tmp.get(&E_int, N));
  cudaMemsetAsync(F_int, 0, sizeof(float) * 3 * N, st);
  cudaMemsetAsync(E_int, 0, sizeof(float) * N, st);
  cudaMemsetAsync(energy_dev, 0, sizeof(double), st);
  double* virial = nullptr;
  if (stress_dev) {
    MLIP_TRY(tmp.get(&virial, 6));
    cudaMemsetAsync(virial, 0, 6 * sizeof(double), st);
  }
  int status = MLIP_OK;
  if (!part) {
    status = mlip_eval_subgraph(ctx, M, L, G->view(), precision, energy_dev, F_int, E_int, virial);
  } else {
    for (size_t k = 0; k < part->subs.size(); ++k) {
      if ((int)(k % (size_t)n_shards) != shard) continue;  // sub-domain k belongs to shard k mod n_shards
      status = mlip_eval_subgraph(ctx, M, L, part->subs[k].g, precision, energy_dev, F_int, E_int, virial);
      if (status != MLIP_OK) break;
    }
  }
  if (status == MLIP_OK && N > 0) {
    k_unpermute<<<nblk(N, 256), 256, 0, st>>>(N, G->perm, F_int, E_int, forces_dev, atom_energy_dev);
    k_check_finite<<<nblk(3 * N, 256), 256, 0, st>>>(3 * N, F_int, energy_dev, ctx->dev_status);
    ctx->launches += 2;
  }
  if (status == MLIP_OK && stress_dev) {
    const double* c = G->cell;
    const double vol = fabs(c[0] * (c[4] * c[8] - c[5] * c[7]) - c[1] * (c[3] * c[8] - c[5] * c[6]) + c[2] * (c[3] * c[7] - c[4] * c[6]));
    k_stress_out<<<1, 32, 0, st>>>(virial, vol > 0.0 ? 1.0 / vol : 0.0, stress_dev);
    ctx->launches++;
  }
  if (status != MLIP_OK) return status;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}

extern "C" int mlip_step_host(mlip_ctx* ctx, const mlip_model* M, int L, const double* pos_host, const double* cell_host,
                              const int32_t* species_host, int64_t N, const int grid[3], double halo, int precision,
                              double* energy_host, float* forces_host) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!M || !pos_host || !cell_host || !species_host || !grid || !energy_host || !forces_host || N < 0) {
    ctx->set_error("mlip_step_host: null argument");
    return MLIP_ERR_INVALID_ARG;
  }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  double *pos_d = nullptr, *e_d = nullptr;
  int32_t* sp_d = nullptr;
  float* f_d = nullptr;
  Scratch tmp(ctx);
  MLIP_TRY(tmp.get(&pos_d, 3 * N)); MLIP_TRY(tmp.get(&sp_d, N)); MLIP_TRY(tmp.get(&f_d, 3 * N));
  MLIP_TRY(tmp.get(&e_d, 1));
  MLIP_CUDA_CHECK(ctx, cudaMemcpyAsync(pos_d, pos_host, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, st));
  MLIP_CUDA_CHECK(ctx, cudaMemcpyAsync(sp_d, species_host, sizeof(int32_t) * N, cudaMemcpyHostToDevice, st));
  mlip_graph* G = nullptr;
  mlip_part* P = nullptr;
  int status = mlip_build_graph(ctx, pos_d, cell_host, sp_d, N, (double)M->h.r_cut, &G);
  if (status == MLIP_OK && (grid[0] > 1 || grid[1] > 1 || grid[2] > 1)) status = mlip_partition_grid(ctx, G, grid, halo, &P);
  if (status == MLIP_OK) status = mlip_energy_forces(ctx, M, L, G, P, precision, e_d, f_d, nullptr);
  if (status == MLIP_OK) {
    cudaMemcpyAsync(energy_host, e_d, sizeof(double), cudaMemcpyDeviceToHost, st);
    cudaMemcpyAsync(forces_host, f_d, sizeof(float) * 3 * N, cudaMemcpyDeviceToHost, st);
  }
  mlip_part_destroy(P);
  mlip_graph_destroy(G);
  cudaError_t e = cudaStreamSynchronize(st);
  if (status != MLIP_OK) return status;
  if (e != cudaSuccess) { ctx->set_error(std::string("step: ") + cudaGetErrorString(e)); return MLIP_ERR_CUDA; }
  return mlip_take_dev_status(ctx);
}
