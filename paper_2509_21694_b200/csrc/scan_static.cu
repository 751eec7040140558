// mlip_scan_i32_noalloc: the exclusive int32 prefix sum of scan.cu (row pointers from degrees, compaction offsets) for
// callers that cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// scan.cu takes its per-tile totals from ctx->alloc; here they live in a file-scope device array of fixed size:
//   g_scan_scratch: MLIP_SCAN_NOALLOC_TILES + 1 int32 = 128 KiB + 4 B per GPU that loads the library, held until exit.
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine: three kernel launches on the
// context stream. Limit: n <= MLIP_SCAN_NOALLOC_MAX = 32768 tiles x 2048 elements = 67,108,864 (config 4 of
// BASELINE.json has 47.2 M edges); larger n is refused with MLIP_ERR_INVALID_ARG.
// Every call on a device SHARES the array and it keeps the previous call's contents. Nothing in it has to start at
// zero (k_sscan_tiles writes every entry the later kernels read), but two calls that overlap on the GPU -- different
// streams, or the same call replayed concurrently from two graphs -- race on it: serialise them.
// mlip_scan_i32 is the same operation through the allocating path the library uses internally (the reference the test of
// this file compares with).
#include <mutex>
#include "common.cuh"

namespace {
constexpr int BS = 256, IPT = 8, TILE = BS * IPT;       // as in scan.cu
constexpr int MAX_TILES = 32768;                        // = 1024 threads x 32 totals of the single-block middle step
constexpr int64_t MAX_N = (int64_t)MAX_TILES * TILE;
static_assert(MAX_N == MLIP_SCAN_NOALLOC_MAX, "include/mlip.h states the limit");

// In host code this name is a host-side stand-in, not a device address: kernels get the pointer that
// cudaGetSymbolAddress returns (scratch_of below).
static __device__ __align__(256) int32_t g_scan_scratch[MAX_TILES + 1];

// block-local exclusive scan of tiles of 2048 elements; tile_sums[tile] = total of the tile
__global__ void __launch_bounds__(BS) k_sscan_tiles(const int32_t* __restrict__ in, int32_t* __restrict__ out,
                                                    int32_t* __restrict__ tile_sums, int64_t n) {
  __shared__ int32_t warp_sums[BS / 32];
  const int64_t base = (int64_t)blockIdx.x * TILE + (int64_t)threadIdx.x * IPT;
  int32_t v[IPT];
  int32_t sum = 0;
#pragma unroll
  for (int k = 0; k < IPT; ++k) {
    v[k] = (base + k < n) ? in[base + k] : 0;
    sum += v[k];
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int32_t incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int32_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int32_t w = lane < BS / 32 ? warp_sums[lane] : 0;
#pragma unroll
    for (int o = 1; o < BS / 32; o <<= 1) {
      const int32_t t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += t;
    }
    if (lane < BS / 32) warp_sums[lane] = w;
  }
  __syncthreads();
  int32_t run = incl - sum + (warp > 0 ? warp_sums[warp - 1] : 0);
#pragma unroll
  for (int k = 0; k < IPT; ++k) {
    if (base + k < n) out[base + k] = run;
    run += v[k];
  }
  if (threadIdx.x == BS - 1) tile_sums[blockIdx.x] = warp_sums[BS / 32 - 1];
}

// ONE block: tile totals -> exclusive tile offsets, in place (thread t owns entries 32 t .. 32 t + 31)
__global__ void __launch_bounds__(1024) k_sscan_offsets(int32_t* __restrict__ sums, int tiles) {
  __shared__ int32_t warp_sums[32];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  int32_t v[32];
  int32_t sum = 0;
#pragma unroll
  for (int k = 0; k < 32; ++k) {
    v[k] = (32 * t + k < tiles) ? sums[32 * t + k] : 0;
    sum += v[k];
  }
  int32_t incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int32_t x = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += x;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int32_t w = warp_sums[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int32_t x = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += x;
    }
    warp_sums[lane] = w;
  }
  __syncthreads();
  int32_t run = incl - sum + (warp > 0 ? warp_sums[warp - 1] : 0);
#pragma unroll
  for (int k = 0; k < 32; ++k) {
    if (32 * t + k < tiles) sums[32 * t + k] = run;
    run += v[k];
  }
}

// out[i] += offset of its tile; out[n] = total
__global__ void k_sscan_add(const int32_t* __restrict__ in, int32_t* __restrict__ out, const int32_t* __restrict__ offs,
                            int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int32_t v = out[i] + offs[i / TILE];
  out[i] = v;
  if (i == n - 1) out[n] = v + in[i];
}
__global__ void k_sscan_empty(int32_t* out) { out[0] = 0; }

// device address of g_scan_scratch, resolved once per device with that device current
int scratch_of(mlip_ctx* ctx, int32_t** out) {
  constexpr int MAX_DEV = 64;
  static std::mutex mu;
  static int32_t* ptr[MAX_DEV] = {nullptr};
  if (ctx->device < 0 || ctx->device >= MAX_DEV) { ctx->set_error("mlip_scan_i32_noalloc: device index out of range"); return MLIP_ERR_INVALID_ARG; }
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[ctx->device]) {
    void* p = nullptr;
    MLIP_CUDA_CHECK(ctx, cudaGetSymbolAddress(&p, g_scan_scratch));
    ptr[ctx->device] = static_cast<int32_t*>(p);
  }
  *out = ptr[ctx->device];
  return MLIP_OK;
}
}  // namespace

extern "C" int mlip_scan_i32_noalloc(mlip_ctx* ctx, const int32_t* in_dev, int32_t* out_dev, int64_t n) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (n < 0 || !out_dev || (n > 0 && !in_dev)) { ctx->set_error("mlip_scan_i32_noalloc: null pointer or negative n"); return MLIP_ERR_INVALID_ARG; }
  if (n > MAX_N) {
    ctx->set_error("mlip_scan_i32_noalloc: n = " + std::to_string(n) + " exceeds MLIP_SCAN_NOALLOC_MAX = " + std::to_string(MAX_N) +
                   " (fixed device scratch of 32768 tile totals); use mlip_scan_i32");
    return MLIP_ERR_INVALID_ARG;
  }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  int32_t* scratch = nullptr;
  MLIP_TRY(scratch_of(ctx, &scratch));
  cudaStream_t st = ctx->stream;
  if (n == 0) {
    k_sscan_empty<<<1, 1, 0, st>>>(out_dev);
    ctx->launches++;
  } else {
    const int tiles = (int)((n + TILE - 1) / TILE);
    k_sscan_tiles<<<(unsigned)tiles, BS, 0, st>>>(in_dev, out_dev, scratch, n);
    k_sscan_offsets<<<1, 1024, 0, st>>>(scratch, tiles);
    k_sscan_add<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in_dev, out_dev, scratch, n);
    ctx->launches += 3;
  }
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}

extern "C" int mlip_scan_i32(mlip_ctx* ctx, const int32_t* in_dev, int32_t* out_dev, int64_t n) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (n < 0 || !out_dev || (n > 0 && !in_dev)) { ctx->set_error("mlip_scan_i32: null pointer or negative n"); return MLIP_ERR_INVALID_ARG; }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  return mlip_exclusive_scan_i32(ctx, in_dev, out_dev, n, nullptr);
}
