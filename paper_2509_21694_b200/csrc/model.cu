// Context + model handles: weight blob upload and the derived operand layouts (transposed /
// sliced fp32 matrices for the CUDA-core path, bf16 operand images for the tcgen05 path).
#include <string.h>
#include "common.cuh"
#include "tc_images.cuh"

namespace {
// dst[r, c] = src[(r0 + (T ? c : r)) * ld + c0 + (T ? r : c)], dst is [rows, cols] dense (ld_dst)
__global__ void k_copy_sub(const float* __restrict__ src, int ld, int r0, int c0, int transpose,
                           float* __restrict__ dst, int ld_dst, int rows, int cols) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= rows * cols) return;
  const int r = idx / cols, c = idx % cols;
  const int sr = r0 + (transpose ? c : r), sc = c0 + (transpose ? r : c);
  dst[(size_t)r * ld_dst + c] = src[(size_t)sr * ld + sc];
}
__global__ void k_scale(const float* __restrict__ src, float* __restrict__ dst, int n, float scale) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = scale * src[i];
}
}  // namespace

extern "C" size_t mlip_model_num_weights(const mlip_model_header* h) {
  if (!h) return 0;
  const size_t S = h->n_species, d = h->d, k = h->n_rbf, L = h->L_max;
  size_t per_layer = d * (2 * d + k) + d + d * d + d + d * 2 * d + d + d * d + d;
  if (h->flags & MLIP_FLAG_THREE_BODY) per_layer += 16 * d + 16 + d * 16;
  return S * d + S + L * per_layer + d * d + d + d + 1;
}

extern "C" int mlip_ctx_create(int device, void* stream, mlip_ctx** out) {
  if (!out) return MLIP_ERR_INVALID_ARG;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
    cudaGetLastError();
    return MLIP_ERR_CUDA;  // no CPU fallback: without a usable device nothing runs
  }
  if (cudaSetDevice(device) != cudaSuccess) return MLIP_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return MLIP_ERR_CUDA;
  if (prop.major != 10) return MLIP_ERR_UNSUPPORTED;  // sm_100a only
  mlip_ctx* c = new mlip_ctx();
  c->device = device;
  c->stream = (cudaStream_t)stream;
  c->num_sms = prop.multiProcessorCount;
  cudaMemPool_t pool;
  if (cudaDeviceGetDefaultMemPool(&pool, device) == cudaSuccess) {
    uint64_t thr = ~0ull;  // keep freed blocks in the pool between steps
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
  }
  if (cudaMalloc((void**)&c->dev_status, sizeof(int)) != cudaSuccess || cudaMemset(c->dev_status, 0, sizeof(int)) != cudaSuccess) {
    cudaGetLastError();
    delete c;
    return MLIP_ERR_OUT_OF_MEMORY;
  }
  *out = c;
  return MLIP_OK;
}

int mlip_take_dev_status(mlip_ctx* ctx) {
  int bits = 0;
  if (cudaMemcpy(&bits, ctx->dev_status, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) {
    ctx->set_error(std::string("status read: ") + cudaGetErrorString(cudaGetLastError()));
    return MLIP_ERR_CUDA;
  }
  if (bits == 0) return MLIP_OK;
  cudaMemset(ctx->dev_status, 0, sizeof(int));
  if (bits & MLIP_DEV_ROW_TOO_LONG) {
    ctx->set_error("three-body variant: an atom has more than 128 neighbours within r_cut3");
    return MLIP_ERR_UNSUPPORTED;
  }
  if (bits & MLIP_DEV_NONFINITE) {
    ctx->set_error("non-finite energy or force: with MLIP_BF16 the edge operands are IEEE half, |pre-activations| and "
                   "|adjoints| must stay below 65504 (use MLIP_FP32 for this model)");
    return MLIP_ERR_NUMERIC;
  }
  ctx->set_error("reverse edge not found while building the graph (internal error)");
  return MLIP_ERR_CUDA;
}

extern "C" int mlip_ctx_status(mlip_ctx* ctx) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) { ctx->set_error(std::string("stream: ") + cudaGetErrorString(e)); return MLIP_ERR_CUDA; }
  return mlip_take_dev_status(ctx);
}

extern "C" void mlip_ctx_destroy(mlip_ctx* ctx) {
  if (!ctx) return;
  cudaFree(ctx->dev_status);
  for (auto& r : ctx->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (cudaEvent_t e : ctx->event_pool) cudaEventDestroy(e);
  delete ctx;
}

static void prof_collect(mlip_ctx* ctx) {
  cudaStreamSynchronize(ctx->stream);
  for (auto& r : ctx->prof) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) {
      ctx->prof_ms[r.cat] += ms;
      ctx->prof_launches[r.cat] += r.launches;
    } else {
      cudaGetLastError();
    }
    ctx->event_pool.push_back(r.a);
    ctx->event_pool.push_back(r.b);
  }
  ctx->prof.clear();
}

extern "C" int mlip_ctx_profile(mlip_ctx* ctx, int enable) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  prof_collect(ctx);
  if (enable) {
    for (int i = 0; i < MLIP_PROF_COUNT; ++i) { ctx->prof_ms[i] = 0.0; ctx->prof_launches[i] = 0; }
  }
  ctx->profiling = enable != 0;
  return MLIP_OK;
}

extern "C" int mlip_ctx_profile_read(mlip_ctx* ctx, int group, double* ms_total, int64_t* n_launches) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (group < 0 || group >= MLIP_PROF_COUNT) { ctx->set_error("unknown kernel group"); return MLIP_ERR_INVALID_ARG; }
  prof_collect(ctx);
  if (ms_total) *ms_total = ctx->prof_ms[group];
  if (n_launches) *n_launches = ctx->prof_launches[group];
  return MLIP_OK;
}
extern "C" const char* mlip_last_error(const mlip_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
extern "C" int64_t mlip_ctx_launch_count(const mlip_ctx* ctx) { return ctx ? ctx->launches : 0; }
extern "C" int mlip_ctx_set_khop_halo(mlip_ctx* ctx, int enable) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  ctx->khop_halo = enable != 0;
  return MLIP_OK;
}
extern "C" int mlip_ctx_set_active_sets(mlip_ctx* ctx, int enable) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  ctx->active_sets = enable != 0;
  return MLIP_OK;
}

extern "C" void mlip_model_destroy(mlip_model* m) {
  if (!m) return;
  for (const void* w : m->x3_keys) m->ctx->x3_img.erase(w);
  for (void* p : m->owned) cudaFree(p);
  delete m;
}

extern "C" int mlip_model_load(mlip_ctx* ctx, const mlip_model_header* h, const float* w_host, size_t n,
                               mlip_model** out) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!h || !w_host || !out) { ctx->set_error("mlip_model_load: null argument"); return MLIP_ERR_INVALID_ARG; }
  *out = nullptr;
  if (h->magic != MLIP_MAGIC || h->version != 1) { ctx->set_error("bad model header magic/version"); return MLIP_ERR_INVALID_ARG; }
  if (h->flags & ~MLIP_FLAG_THREE_BODY) { ctx->set_error("unknown model flags"); return MLIP_ERR_UNSUPPORTED; }
  if (h->flags & MLIP_FLAG_THREE_BODY) {
    if (h->n_rbf3 != 4 || h->l_max != 3 || !(h->r_cut3 > 0.f) || h->r_cut3 > h->r_cut) {
      ctx->set_error("three-body variant needs n_rbf3 = 4, l_max = 3 and 0 < r_cut3 <= r_cut");
      return MLIP_ERR_UNSUPPORTED;
    }
  } else if (h->n_rbf3 != 0 || h->l_max != 0 || h->r_cut3 != 0.f) {
    ctx->set_error("n_rbf3, l_max and r_cut3 must be 0 without MLIP_FLAG_THREE_BODY");
    return MLIP_ERR_INVALID_ARG;
  }
  if (!(h->d == 64 || h->d == 128 || h->d == 256) || h->n_rbf < 2 || h->n_rbf > 16 || h->n_species < 1 ||
      h->L_max < 0 || !(h->r_cut > 0.f)) {
    ctx->set_error("unsupported model shape (d in {64,128,256}, 2 <= n_rbf <= 16)");
    return MLIP_ERR_UNSUPPORTED;
  }
  if (n != mlip_model_num_weights(h)) { ctx->set_error("weight blob size does not match header"); return MLIP_ERR_INVALID_ARG; }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  mlip_model* M = new mlip_model();
  M->h = *h; M->ctx = ctx;
  const int S = h->n_species, d = h->d, k = h->n_rbf, L = h->L_max;
  auto fail = [&](int code) { mlip_model_destroy(M); return code; };
  auto dalloc = [&](size_t bytes) -> void* {
    void* p = nullptr;
    if (cudaMalloc(&p, bytes ? bytes : 1) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    M->owned.push_back(p);
    return p;
  };
#define M_ALLOC(ptr, T, count)                                                         \
  do {                                                                                 \
    ptr = (T*)dalloc(sizeof(T) * (size_t)(count));                                     \
    if (!ptr) { ctx->set_error("out of device memory (model)"); return fail(MLIP_ERR_OUT_OF_MEMORY); } \
  } while (0)
  // Device copy of the blob with every tensor on a 16-byte boundary: the kernels read weights as float4, and the
  // offsets inside the caller's blob are arbitrary (E0 has S floats).
  const size_t n_tensors = 2 + (size_t)L * 11 + 4;
  M_ALLOC(M->blob, float, n + 4 * n_tensors);
  size_t src_off = 0, dst_off = 0;
  bool upload_ok = true;
  auto take = [&](size_t count) -> const float* {
    dst_off = (dst_off + 3) & ~(size_t)3;
    float* dst = M->blob + dst_off;
    if (cudaMemcpyAsync(dst, w_host + src_off, count * sizeof(float), cudaMemcpyHostToDevice, st) != cudaSuccess) upload_ok = false;
    src_off += count; dst_off += count;
    return dst;
  };
  M->T = take((size_t)S * d);
  M->E0 = take(S);
  M->layers.resize(L);
  auto sub = [&](const float* src, int ld, int r0, int c0, int tr, float* dst, int ld_dst, int rows, int cols) {
    k_copy_sub<<<(rows * cols + 255) / 256, 256, 0, st>>>(src, ld, r0, c0, tr, dst, ld_dst, rows, cols);
  };
  // bf16 SWIZZLE_128B operand image of a row-major [N, K] weight (node_bf16.cu streams it slab by slab)
  auto toimg = [&](const float* src, mlip_nodeop* dst, int N, int K, float scale = 1.0f) {
    mlip_make_gemm_image(st, src, N, K, scale, dst);
  };
  for (int l = 0; l < L; ++l) {
    LayerWeights& W = M->layers[l];
    memset(&W, 0, sizeof(W));
    W.W1 = take((size_t)d * (2 * d + k));
    W.b1 = take(d);
    W.W2 = take((size_t)d * d);
    W.b2 = take(d);
    W.V1 = take((size_t)d * 2 * d);
    W.c1 = take(d);
    W.V2 = take((size_t)d * d);
    W.c2 = take(d);
    if (h->flags & MLIP_FLAG_THREE_BODY) {
      W.G3 = take((size_t)16 * d);
      W.g3 = take(16);
      W.W3 = take((size_t)d * 16);
    }
    M_ALLOC(W.W1ab, float, 2 * d * d); M_ALLOC(W.W1c, float, d * 16); M_ALLOC(W.W1abT, float, 2 * d * d);
    M_ALLOC(W.W2T, float, d * d); M_ALLOC(W.V2T, float, d * d); M_ALLOC(W.V1aT, float, d * d);
    M_ALLOC(W.V1bT, float, d * d); M_ALLOC(W.b1pad, float, 2 * d);
    const int ld1 = 2 * d + k;
    sub(W.W1, ld1, 0, 0, 0, W.W1ab, d, d, d);                    // W1a
    sub(W.W1, ld1, 0, d, 0, W.W1ab + (size_t)d * d, d, d, d);    // W1b
    cudaMemsetAsync(W.W1c, 0, sizeof(float) * d * 16, st);
    sub(W.W1, ld1, 0, 2 * d, 0, W.W1c, 16, d, k);                // W1c padded to 16 columns
    sub(W.W1, ld1, 0, 0, 1, W.W1abT, 2 * d, d, d);               // W1a^T
    sub(W.W1, ld1, 0, d, 1, W.W1abT + d, 2 * d, d, d);           // W1b^T
    sub(W.W2, d, 0, 0, 1, W.W2T, d, d, d);
    sub(W.V2, d, 0, 0, 1, W.V2T, d, d, d);
    sub(W.V1, 2 * d, 0, 0, 1, W.V1aT, d, d, d);
    sub(W.V1, 2 * d, 0, d, 1, W.V1bT, d, d, d);
    cudaMemsetAsync(W.b1pad, 0, sizeof(float) * 2 * d, st);
    cudaMemcpyAsync(W.b1pad, W.b1, sizeof(float) * d, cudaMemcpyDeviceToDevice, st);
    // bf16 operand images for the tensor-core node GEMMs (B operands are [N, K])
    M_ALLOC(W.W1a_bf, mlip_nodeop, d * d); M_ALLOC(W.W1b_bf, mlip_nodeop, d * d);
    M_ALLOC(W.V1_bf, mlip_nodeop, 2 * d * d); M_ALLOC(W.V2_bf, mlip_nodeop, d * d);
    M_ALLOC(W.V2T_bf, mlip_nodeop, d * d); M_ALLOC(W.V1aT_bf, mlip_nodeop, d * d);
    M_ALLOC(W.V1bT_bf, mlip_nodeop, d * d); M_ALLOC(W.W1abT_bf, mlip_nodeop, 2 * d * d);
    // the tensor-core edge kernels consume HALVED pre-projections P' = (W1a h + b1)/2, Q' = (W1b h)/2 (exact scaling)
    toimg(W.W1ab, W.W1a_bf, d, d, 0.5f); toimg(W.W1ab + (size_t)d * d, W.W1b_bf, d, d, 0.5f);
    M_ALLOC(W.b1h, float, d);
    k_scale<<<(d + 255) / 256, 256, 0, st>>>(W.b1, W.b1h, d, 0.5f);
    toimg(W.V1, W.V1_bf, d, 2 * d); toimg(W.V2, W.V2_bf, d, d); toimg(W.V2T, W.V2T_bf, d, d);
    toimg(W.V1aT, W.V1aT_bf, d, d); toimg(W.V1bT, W.V1bT_bf, d, d); toimg(W.W1abT, W.W1abT_bf, d, 2 * d);
    // operand images of the fused edge kernels (tc_images.cuh documents the layouts)
    M_ALLOC(W.W2img, __half, d * d); M_ALLOC(W.W1cimg, __half, d * 16);
    mlip_make_edge_images(st, W.W2, W.W1c, d, W.W2img, W.W1cimg);
    if (d == 128) {
      M_ALLOC(W.W2x3, __nv_bfloat16, 3 * d * d); M_ALLOC(W.W13x3, __nv_bfloat16, 3 * d * 32);
      mlip_make_edge_images_x3(st, W.W2, W.W1c, W.W3, d, W.W2x3, W.W13x3);
    }
  }
  M->Wo = take((size_t)d * d);
  M->bo = take(d);
  M->wo = take(d);
  M->bE = take(1);
  if (!upload_ok || src_off != n) { ctx->set_error("weight upload failed"); return fail(MLIP_ERR_CUDA); }
  M_ALLOC(M->WoT, float, d * d);
  sub(M->Wo, d, 0, 0, 1, M->WoT, d, d, d);
  M_ALLOC(M->Wo_bf, mlip_nodeop, d * d); M_ALLOC(M->WoT_bf, mlip_nodeop, d * d);
  toimg(M->Wo, M->Wo_bf, d, d); toimg(M->WoT, M->WoT_bf, d, d);
  if (d == 128) {
    // three-term bf16 split images of every weight matrix the fp32 node GEMMs multiply by (node_x3.cu)
    auto img3 = [&](const float* Wm, int N, int K) -> int {
      __nv_bfloat16* img = nullptr;
      M_ALLOC(img, __nv_bfloat16, 3 * (size_t)N * K);
      mlip_make_gemm_image_x3(st, Wm, N, K, img);
      ctx->x3_img[Wm] = img;
      M->x3_keys.push_back(Wm);
      return MLIP_OK;
    };
    for (int l = 0; l < L; ++l) {
      LayerWeights& W = M->layers[l];
      MLIP_TRY(img3(W.W1ab, 2 * d, d)); MLIP_TRY(img3(W.V1, d, 2 * d)); MLIP_TRY(img3(W.V2, d, d)); MLIP_TRY(img3(W.V2T, d, d));
      MLIP_TRY(img3(W.V1aT, d, d)); MLIP_TRY(img3(W.V1bT, d, d)); MLIP_TRY(img3(W.W1abT, d, 2 * d));
    }
    MLIP_TRY(img3(M->Wo, d, d)); MLIP_TRY(img3(M->WoT, d, d));
  }
#undef M_ALLOC
  if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
    ctx->set_error("model preparation kernels failed");
    return fail(MLIP_ERR_CUDA);
  }
  *out = M;
  return MLIP_OK;
}
