// Argument block and launchers of the fused edge kernels (fp32 CUDA-core and bf16 tcgen05 paths).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include "common.cuh"

struct EdgeArgs {
  int64_t E = 0, n = 0;
  // Verlet-skin mode of the MD driver: the edge list is re-filtered on the device every step, so its length is only known
  // there. When given, the number of edges is *E_dyn (= rowptr[number of receivers of this launch]) and E above is the
  // CAPACITY the launch dimensions are derived from (fixed between rebuilds, which is what lets a CUDA graph replay them).
  const int32_t* E_dyn = nullptr;
  const int32_t* rowptr = nullptr;
  const int32_t* recv = nullptr;
  const int32_t* send = nullptr;
  const int32_t* rev = nullptr;
  const float4* rvec = nullptr;
  const float* P = nullptr; int ldp = 0;           // receiver pre-projection W1a h_i + b1 (fp32 path)
  const __half* Ph = nullptr;                      // halved receiver pre-projection (tensor-core path, f16), ld = d
  const float* Q = nullptr; int ldq = 0;           // sender pre-projection W1b h_j (fp32 path)
  const __half* Qh = nullptr;                      // halved sender pre-projection (tensor-core path, f16), ld = d
  // tensor-core path: when given, row a of Ph / Qh belongs to atom i with row_index[i] == a. The first layer passes the
  // species here: h^0 is the species embedding, so P^0 and Q^0 are S-row tables and the per-edge gathers hit L1
  const int32_t* row_index = nullptr;
  const float* W1c = nullptr;                      // [d,16] fp32
  const float* W2T = nullptr;                      // [in,out] fp32
  const float* W2 = nullptr;                       // [out,in] fp32
  const __half *W2img = nullptr, *W1cimg = nullptr;  // f16 operand images, tc_images.cuh
  // fp32 path on the tensor cores (edge_x3.cu, d = 128): three-term bf16 split images of W2 and of [W1c | W3], or null
  const __nv_bfloat16 *W2x3 = nullptr, *W13x3 = nullptr;
  const float* b2 = nullptr;
  float r_cut = 0.f, alpha = 0.f;
  int n_rbf = 0;
  float* m = nullptr;                              // forward out [n,d]
  float *head = nullptr, *tail = nullptr;          // per-tile partial rows [tiles,d]
  const float* mbar = nullptr;                     // backward in [n,d] (fp32 path)
  const __half* mbar_h = nullptr;                  // backward in [n,d] (tensor-core path, f16)
  float* abar = nullptr;                           // backward spill [E,d] fp32
  __half* abar_h = nullptr;                        // backward spill, f16 tile images [tiles,128,d]
  float* Pbar = nullptr;                           // backward out [n,d]
  float* rbar = nullptr;                           // [E] accumulated over layers
  // backward only: false for the FIRST layer, whose node-side adjoints (Pbar, the spilled abar -> Qbar) would only feed
  // the gradient w.r.t. the species embedding -- forces need nothing but rbar, so the spill, the segmented sum and the
  // sender-side gather of that layer are skipped
  bool node_adjoint = true;
  // three-body variant (fp32 path): a_e += W3 t_e; the reverse pass writes tbar_e = W3^T abar_e
  const float* t3 = nullptr;    // [E,16] or null
  const float* W3 = nullptr;    // [d,16]
  float* tbar = nullptr;        // [E,16] (backward out)
};

// three_body.cu
int mlip_gate_forward(mlip_ctx* ctx, int64_t n, int d, const float* h, const float* G, const float* g, float* z);
int mlip_triplet_forward(mlip_ctx* ctx, int64_t n_recv, float r3, const int32_t* rowptr, const int32_t* send,
                         const float4* rvec, const float* z, float* t, int* long_rows /* scratch, int[n_recv + 1] */);
int mlip_triplet_backward(mlip_ctx* ctx, int64_t n_recv, float r3, const int32_t* rowptr, const int32_t* send,
                          const float4* rvec, const float* z, const float* tbar, float* rbar, float4* gvec, float* zeta,
                          int* long_rows /* scratch, int[n_recv + 1] */);
int mlip_gate_backward(mlip_ctx* ctx, int64_t n_send, int64_t E_act, const int32_t* E_act_dyn, int d, const int32_t* rowptr,
                       const int32_t* rev, const float* zeta, const float* z, const float* G, float* hbar);

int64_t mlip_edge_f32_tiles(int64_t E);
int mlip_edge_forward_f32(mlip_ctx* ctx, int d, const EdgeArgs& a);
int mlip_edge_backward_f32(mlip_ctx* ctx, int d, const EdgeArgs& a);
// Qbar_j = sum over in-edges e of j, j < n, with rev[e] < E_act, of abar[rev[e]]
int mlip_gather_rev_f32(mlip_ctx* ctx, int64_t n, int64_t E_act, const int32_t* E_act_dyn, int d, const int32_t* rowptr,
                        const int32_t* rev, const float* abar, float* Qbar);

// fp32 operands split into three bf16 terms on tcgen05 (d = 128; mlip_edge_*_f32 dispatch to it)
bool mlip_edge_x3_supported(int d, const EdgeArgs& a);
int mlip_edge_forward_x3(mlip_ctx* ctx, const EdgeArgs& a);
int mlip_edge_backward_x3(mlip_ctx* ctx, const EdgeArgs& a);

int64_t mlip_edge_tc_tiles(int64_t E);
int mlip_edge_forward_tc(mlip_ctx* ctx, int d, const EdgeArgs& a);
int mlip_edge_backward_tc(mlip_ctx* ctx, int d, const EdgeArgs& a);
int mlip_gather_rev_tc(mlip_ctx* ctx, int64_t n, int64_t E_act, const int32_t* E_act_dyn, int d, const int32_t* rowptr,
                       const int32_t* rev, const __half* abar, mlip_nodeop* Qbar /*[n,d] bf16*/);
