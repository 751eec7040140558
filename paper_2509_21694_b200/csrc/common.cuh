// Shared host-side definitions of the mlip B200 library: context, handles, error plumbing and
// the declarations of the kernel launchers implemented in the other translation units.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <string>
#include <unordered_map>
#include <vector>
#include "../../include/mlip.h"

// 16-bit operand type of the node contractions (see tc_ptx.cuh): IEEE half unless MLIP_NODE_OPERANDS_BF16
#ifdef MLIP_NODE_OPERANDS_BF16
typedef __nv_bfloat16 mlip_nodeop;
#else
typedef __half mlip_nodeop;
#endif

#define MLIP_CUDA_CHECK(ctx, expr)                                                        \
  do {                                                                                    \
    cudaError_t _e = (expr);                                                              \
    if (_e != cudaSuccess) {                                                              \
      (ctx)->set_error(std::string(#expr) + ": " + cudaGetErrorString(_e));               \
      return _e == cudaErrorMemoryAllocation ? MLIP_ERR_OUT_OF_MEMORY : MLIP_ERR_CUDA;    \
    }                                                                                     \
  } while (0)

#define MLIP_TRY(expr)              \
  do {                              \
    int _s = (expr);                \
    if (_s != MLIP_OK) return _s;   \
  } while (0)

// kernel groups timed by mlip_ctx_profile (CUDA events on the context stream)
enum {
  MLIP_PROF_EDGE_FWD = 0,   // fused gather -> edge MLP -> segmented sum (A6+A7)
  MLIP_PROF_EDGE_BWD = 1,   // its reverse pass (edge part of A10)
  MLIP_PROF_GATHER_REV = 2, // sender-side adjoint gather through rev[]
  MLIP_PROF_NODE_GEMM = 3,  // node pre-projection / node update / readout GEMMs and adjoints
  MLIP_PROF_READOUT_FORCES = 4,  // embedding, readout, energy sum, force assembly
  MLIP_PROF_GRAPH = 5,      // mlip_build_graph
  MLIP_PROF_PARTITION = 6,  // mlip_partition*
  MLIP_PROF_THREE_BODY = 7, // gate, triplet and their adjoint kernels of the three-body variant
  MLIP_PROF_COUNT = 8
};

struct mlip_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int num_sms = 148;
  std::string err;
  int64_t launches = 0;
  bool active_sets = true;  // per-layer active sets inside sub-domains (mlip_ctx_set_active_sets)
  bool khop_halo = true;    // halo and depth classes by K-hop search instead of geometry (mlip_ctx_set_khop_halo)
  // Sticky device-side status word (MLIP_DEV_* bits, written by kernels with atomicOr): errors that only the device can
  // see (non-finite results of the 16-bit path, a missing reverse edge) surface at the next synchronising call or at
  // mlip_ctx_status, never as silently wrong numbers.
  int* dev_status = nullptr;
  // fp32 weight matrix (device pointer, the GemmArgs::B of the fp32 path) -> its three-term bf16 split image for the
  // tensor-core fp32 node GEMM (node_x3.cu); filled by mlip_model_load at d = 128, emptied by mlip_model_destroy
  std::unordered_map<const void*, const __nv_bfloat16*> x3_img;
  void set_error(const std::string& s) { err = s; }
  // ---- optional per-group timing ----
  struct ProfRec { int cat; int64_t launches; cudaEvent_t a, b; };
  bool profiling = false;
  std::vector<ProfRec> prof;
  std::vector<cudaEvent_t> event_pool;
  double prof_ms[MLIP_PROF_COUNT] = {0};
  int64_t prof_launches[MLIP_PROF_COUNT] = {0};
  cudaEvent_t get_event() {
    cudaEvent_t e;
    if (!event_pool.empty()) { e = event_pool.back(); event_pool.pop_back(); return e; }
    cudaEventCreate(&e);
    return e;
  }
  // returns a token (index + 1) or 0 when profiling is off
  size_t prof_begin(int cat) {
    if (!profiling) return 0;
    ProfRec r; r.cat = cat; r.launches = launches; r.a = get_event(); r.b = get_event();
    cudaEventRecord(r.a, stream);
    prof.push_back(r);
    return prof.size();
  }
  void prof_end(size_t token) {
    if (!token) return;
    ProfRec& r = prof[token - 1];
    r.launches = launches - r.launches;
    cudaEventRecord(r.b, stream);
  }
  // stream-ordered allocation (pool keeps memory between steps)
  template <class T>
  int alloc(T** p, size_t n) {
    *p = nullptr;
    if (n == 0) n = 1;
    cudaError_t e = cudaMallocAsync((void**)p, n * sizeof(T), stream);
    if (e != cudaSuccess) {
      set_error(std::string("cudaMallocAsync: ") + cudaGetErrorString(e));
      cudaGetLastError();
      return MLIP_ERR_OUT_OF_MEMORY;
    }
    return MLIP_OK;
  }
  void free(void* p) {
    if (p) cudaFreeAsync(p, stream);
  }
};

enum { MLIP_DEV_REV_MISSING = 1, MLIP_DEV_NONFINITE = 2, MLIP_DEV_ROW_TOO_LONG = 4 };
// Reads and clears the device status word; the stream must have been synchronised. Returns MLIP_OK or the status the
// bits map to (with the context error message set).
int mlip_take_dev_status(mlip_ctx* ctx);

// Stream-ordered scratch buffers that are released when the scope ends, on every path out of it.
struct Scratch {
  mlip_ctx* c;
  std::vector<void*> v;
  explicit Scratch(mlip_ctx* ctx) : c(ctx) {}
  ~Scratch() { for (void* p : v) c->free(p); }
  template <class T>
  int get(T** p, size_t n) {
    const int s = c->alloc(p, n);
    if (s == MLIP_OK) v.push_back(*p);
    return s;
  }
};

struct ProfScope {
  mlip_ctx* c; size_t t;
  ProfScope(mlip_ctx* ctx, int cat) : c(ctx), t(ctx->prof_begin(cat)) {}
  ~ProfScope() { c->prof_end(t); }
};

// ---- model --------------------------------------------------------------------------------
struct LayerWeights {
  // fp32 device pointers into the blob copy (row-major [out,in])
  const float *W1, *b1, *W2, *b2, *V1, *c1, *V2, *c2;
  const float *G3 = nullptr, *g3 = nullptr, *W3 = nullptr;  // three-body variant: G[16,d], g[16], W3[d,16] (blob)
  // derived fp32 matrices (device, owned by the model)
  float* W1ab;    // [2d, d]  rows 0..d-1 = W1a (receiver block), d..2d-1 = W1b (sender block)
  float* W1c;     // [d, n_rbf]
  float* W1abT;   // [d, 2d]  = [W1a^T | W1b^T]   (backward: hbar += Pbar W1a + Qbar W1b)
  float* W2T;     // [d, d]   W2 transposed ([in,out])
  float* V2T;     // [d, d]
  float* V1aT;    // [d, d]   (V1[:, :d])^T
  float* V1bT;    // [d, d]   (V1[:, d:])^T
  float* b1pad;   // [2d] = [b1 | 0]
  float* b1h;     // [d] = b1 / 2 (bias of the halved receiver pre-projection of the bf16 path)
  // bf16 operand images for the tensor-core path (device, owned); see tc_common.cuh
  __half *W2img, *W1cimg;
  __nv_bfloat16 *W2x3 = nullptr, *W13x3 = nullptr;  // three-term split images of the fp32 tensor-core edge kernels (d = 128)
  mlip_nodeop *W1a_bf, *W1b_bf, *V1_bf, *V2_bf, *V2T_bf, *V1aT_bf, *V1bT_bf, *W1abT_bf;
};

struct mlip_model {
  mlip_model_header h;
  mlip_ctx* ctx;
  float* blob = nullptr;  // device copy of the caller's blob
  const float *T, *E0, *Wo, *bo, *wo, *bE;
  float* WoT = nullptr;   // [d,d]
  mlip_nodeop *Wo_bf = nullptr, *WoT_bf = nullptr;
  std::vector<LayerWeights> layers;
  std::vector<void*> owned;  // everything to cudaFree
  std::vector<const void*> x3_keys;  // this model's entries of mlip_ctx::x3_img
};

// ---- graph --------------------------------------------------------------------------------
constexpr int MLIP_MAX_CLS = 32;
// A (sub)graph in the form the model kernels consume: atoms are numbered locally, edges are
// sorted by receiver, rows sorted by (sender, shift).
struct SubGraph {
  int64_t n = 0;        // atoms (extended set)
  int64_t n_owned = 0;  // root atoms
  int64_t E = 0;        // directed edges
  const int32_t* gid = nullptr;    // [n] index into the graph's internal numbering (nullptr = identity)
  const float* omega = nullptr;    // [n] 1 for root atoms, 0 for halo atoms (nullptr = all ones)
  const int32_t* species = nullptr;  // [n]
  const int32_t* rowptr = nullptr;   // [n+1]
  const int32_t* recv = nullptr;     // [E]
  const int32_t* send = nullptr;     // [E]
  const int32_t* rev = nullptr;      // [E] index of the reverse edge
  const float4* rvec = nullptr;      // [E] (r_x, r_y, r_z, |r|), float32 rounded from float64
  // Depth classes (sub-domains only; n_cls == 0 means "no classes, every layer runs on all atoms"). Atoms are numbered
  // by (class, cell order): class 0 = root atoms, class k >= 1 = halo atoms k hops from the nearest root atom (K-hop
  // search) or, geometric variant, whose largest per-axis periodic distance to the bin lies in ((k-1) r_c, k r_c]. Either
  // way an atom of class k only has neighbours of class >= k-1, so the root energies (and their gradient) need layer l
  // only on receivers of class <= L-1-l with senders of class <= L-l (each root atom keeps its K-hop
  // neighbourhood). Both sets are prefixes of the numbering.
  // Verlet-skin mode (md.cu / skin.cu): the edge arrays are re-filtered on the device every step; E and E_le are then
  // CAPACITIES (the candidate counts) and the actual numbers are rowptr[n] / rowptr[n_le[c]] on the device.
  bool dyn = false;
  int n_cls = 0;
  int64_t n_le[MLIP_MAX_CLS] = {};   // atoms of class <= c
  int64_t E_le[MLIP_MAX_CLS] = {};   // edges whose receiver has class <= c  (= rowptr[n_le[c]])
  int64_t atoms_upto(int c) const { return n_cls == 0 ? n : n_le[c < 0 ? 0 : (c >= n_cls ? n_cls - 1 : c)]; }
  int64_t edges_upto(int c) const { return n_cls == 0 ? E : E_le[c < 0 ? 0 : (c >= n_cls ? n_cls - 1 : c)]; }
};

struct mlip_graph {
  mlip_ctx* ctx;
  int64_t N = 0, E = 0;
  double cell[9], inv[9], width[3];
  double r_cut = 0;
  int nc[3];
  int32_t* perm = nullptr;      // [N] internal -> caller index
  double* frac = nullptr;       // [N,3] wrapped fractional coordinates, internal order
  int32_t* species = nullptr;   // [N] internal order
  int species_min = 0, species_max = 0;  // range of the species values (read back with the edge count)
  int32_t* rowptr = nullptr;    // [N+1]
  int32_t* recv = nullptr;      // [E]
  int32_t* send = nullptr;      // [E]
  int32_t* shift = nullptr;     // [E] packed (nx+128)<<16 | (ny+128)<<8 | (nz+128)
  int32_t* rev = nullptr;       // [E]
  float4* rvec = nullptr;       // [E]
  SubGraph view() const {
    SubGraph s;
    s.n = N; s.n_owned = N; s.E = E; s.species = species; s.rowptr = rowptr; s.recv = recv;
    s.send = send; s.rev = rev; s.rvec = rvec;
    return s;
  }
};

struct PartSub {
  SubGraph g;
  int32_t *gid = nullptr, *species = nullptr, *rowptr = nullptr, *recv = nullptr, *send = nullptr,
          *rev = nullptr;
  float* omega = nullptr;
  float4* rvec = nullptr;
  int32_t* geid = nullptr;   // [E] edge id in the parent graph (kept on request: mlip_partition_grid_ex)
};

struct mlip_part {
  mlip_ctx* ctx;
  int grid[3];
  double halo = 0;
  bool khop = false;  // classes are hop counts (K-hop search) rather than geometric shells
  int64_t N = 0;
  int shard = 0, n_shards = 1;  // mlip_partition_grid_shard: only sub-domains k with k mod n_shards == shard were built
  std::vector<PartSub> subs;
};

int mlip_partition_grid_ex(mlip_ctx* ctx, const mlip_graph* G, const int grid[3], double halo_box, double halo,
                           double r_class, bool force_khop, bool keep_geid, mlip_part** out, int shard = 0, int n_shards = 1);

// ---- launchers (each bumps ctx->launches by the number of kernels it enqueues) ---------------
// scan.cu
int mlip_exclusive_scan_i32(mlip_ctx* ctx, const int32_t* in, int32_t* out, int64_t n,
                            int64_t* total_host /*nullable; synchronises when given*/);

// node_f32.cu -- Y[n,N] = epi( act(X)[n,K] . B^T + bias ), X = [X1 | X2] column blocks
struct GemmArgs {
  const float* X1 = nullptr; int ld1 = 0; int K1 = 0;
  const float* X2 = nullptr; int ld2 = 0; int K2 = 0;
  // tensor-core path only: a column block may be given as bf16 instead (same ld / K fields); it is then copied
  // into the operand slab as it is -- the value the fp32 form would have been rounded to on load
  const mlip_nodeop* X1b = nullptr;
  const mlip_nodeop* X2b = nullptr;
  int act_in = 0;                 // 1: SiLU applied to X on load
  const void* B = nullptr;        // [N, K1+K2] row-major (fp32 path) / bf16 SW128 operand image (tensor path)
  const float* bias = nullptr;    // [N]
  const float* mul_dsilu = nullptr; int ldz = 0;  // epilogue: y *= SiLU'(Z[row, col])
  const float* residual = nullptr; int ldr = 0;   // epilogue: y += R[row, col] (may alias Y)
  float* Y = nullptr; int ldy = 0;                // fp32 output (or)
  mlip_nodeop* Ybf = nullptr;                   // bf16 output (same ldy)
  __half* Yh = nullptr;                           // f16 output (same ldy)
  int64_t n = 0; int N = 0;
};
int mlip_gemm_f32(mlip_ctx* ctx, const GemmArgs& a);
// node_x3.cu: the fp32 GEMM on tcgen05 with 3-term bf16 operand splits (mlip_gemm_f32 dispatches to it when B has an image)
void mlip_make_gemm_image_x3(cudaStream_t st, const float* W, int N, int K, __nv_bfloat16* img /*[3][N*K]*/);
bool mlip_gemm_x3_supported(const GemmArgs& a);
int mlip_gemm_x3(mlip_ctx* ctx, const GemmArgs& a, const __nv_bfloat16* Bx3);
int mlip_gemm_bf16(mlip_ctx* ctx, const GemmArgs& a);  // B = image built by mlip_make_gemm_image
void mlip_make_gemm_image(cudaStream_t st, const float* W, int N, int K, float scale, mlip_nodeop* img);

// energy_forces.cu
int mlip_eval_subgraph(mlip_ctx* ctx, const mlip_model* m, int L, const SubGraph& g, int precision,
                       double* energy_accum_dev, float* forces_internal /*[N,3]*/,
                       float* atom_energy_internal /*[N] or null*/,
                       double* virial_accum_dev /*[6] xx,yy,zz,yz,xz,xy or null*/);
