// Exclusive prefix sum over int32 (cell counts, degrees, compaction flags): block-local scan,
// recursive scan of the block totals, offset add. Plain integer work; results are exact.
#include "common.cuh"

namespace {
constexpr int SCAN_BS = 256;
constexpr int SCAN_IPT = 8;
constexpr int SCAN_TILE = SCAN_BS * SCAN_IPT;

__global__ void __launch_bounds__(SCAN_BS) k_scan_tiles(const int32_t* __restrict__ in,
                                                         int32_t* __restrict__ out,
                                                         int32_t* __restrict__ tile_sums, int64_t n) {
  __shared__ int32_t warp_sums[SCAN_BS / 32];
  const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_IPT;
  int32_t v[SCAN_IPT];
  int32_t sum = 0;
#pragma unroll
  for (int k = 0; k < SCAN_IPT; ++k) {
    v[k] = (base + k < n) ? in[base + k] : 0;
    sum += v[k];
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int32_t incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int32_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int32_t w = lane < SCAN_BS / 32 ? warp_sums[lane] : 0;
#pragma unroll
    for (int o = 1; o < SCAN_BS / 32; o <<= 1) {
      int32_t t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += t;
    }
    if (lane < SCAN_BS / 32) warp_sums[lane] = w;  // inclusive over warps
  }
  __syncthreads();
  int32_t run = incl - sum + (warp > 0 ? warp_sums[warp - 1] : 0);
#pragma unroll
  for (int k = 0; k < SCAN_IPT; ++k) {
    if (base + k < n) out[base + k] = run;
    run += v[k];
  }
  if (threadIdx.x == SCAN_BS - 1) tile_sums[blockIdx.x] = warp_sums[SCAN_BS / 32 - 1];
}

__global__ void k_scan_add(int32_t* __restrict__ out, const int32_t* __restrict__ tile_offs, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] += tile_offs[i / SCAN_TILE];
}

__global__ void k_scan_total(int32_t* out, const int32_t* in, int64_t n) {
  // out[n] = out[n-1] + in[n-1]
  if (threadIdx.x == 0 && blockIdx.x == 0) out[n] = n > 0 ? out[n - 1] + in[n - 1] : 0;
}
}  // namespace

static int scan_rec(mlip_ctx* ctx, const int32_t* in, int32_t* out, int64_t n) {
  if (n <= 0) return MLIP_OK;
  const int64_t tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  int32_t* sums = nullptr;
  MLIP_TRY(ctx->alloc(&sums, (size_t)tiles + 1));
  k_scan_tiles<<<(unsigned)tiles, SCAN_BS, 0, ctx->stream>>>(in, out, sums, n);
  ctx->launches++;
  if (tiles > 1) {
    int32_t* offs = nullptr;
    MLIP_TRY(ctx->alloc(&offs, (size_t)tiles + 1));
    MLIP_TRY(scan_rec(ctx, sums, offs, tiles));
    k_scan_add<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(out, offs, n);
    ctx->launches++;
    ctx->free(offs);
  }
  ctx->free(sums);
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}

// out has n+1 entries; out[n] = total. `in` and `out` must not alias.
int mlip_exclusive_scan_i32(mlip_ctx* ctx, const int32_t* in, int32_t* out, int64_t n,
                            int64_t* total_host) {
  MLIP_TRY(scan_rec(ctx, in, out, n));
  k_scan_total<<<1, 32, 0, ctx->stream>>>(out, in, n);
  ctx->launches++;
  if (total_host) {
    int32_t t = 0;
    MLIP_CUDA_CHECK(ctx, cudaMemcpyAsync(&t, out + n, sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
    MLIP_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    *total_host = t;
  }
  return MLIP_OK;
}
