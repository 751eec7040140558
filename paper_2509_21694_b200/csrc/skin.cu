// Verlet-skin reuse of the radius graph and of the partition in the MD driver (PAPER.md:89, 131 run
// 10^5..10^6-step trajectories, PAPER.md:165 wants graph + partition below 2 % of a step). The candidate list -- the
// radius graph at r_c + skin, partitioned once -- stays fixed between rebuilds; every step it is FILTERED with the
// canonical float64 predicate of O1 at the current positions, which yields exactly the edge set (and, rows being sorted
// subsets of sorted rows, exactly the order) a fresh mlip_build_graph would give as long as no atom has moved more than
// skin/2. All launch dimensions depend on the candidate sizes only; the filtered sizes stay on the device
// (SubGraph::dyn), so the whole step can be replayed from a CUDA graph.
#include "canon.cuh"
#include "common.cuh"
#include "skin.cuh"

namespace {
inline unsigned nblk(int64_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// candidate shifts / caller atom ids of a sub-domain from its parent graph
__global__ void k_skin_gather_sub(int64_t n, int64_t E, const int32_t* __restrict__ gid, const int32_t* __restrict__ perm,
                                  const int32_t* __restrict__ geid, const int32_t* __restrict__ g_shift,
                                  int32_t* __restrict__ aid, int32_t* __restrict__ c_shift) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) aid[i] = perm[gid ? gid[i] : i];
  if (i < E) c_shift[i] = geid ? g_shift[geid[i]] : g_shift[i];
}

struct Cell9 { double c[9]; };

// pass 1: which candidates of row l are edges at the current positions; rank inside the row, row length
__global__ void __launch_bounds__(256) k_skin_count(int64_t n, const int32_t* __restrict__ c_rowptr,
                                                    const int32_t* __restrict__ c_send, const int32_t* __restrict__ c_shift,
                                                    const int32_t* __restrict__ aid, const double* __restrict__ pos, Cell9 cell,
                                                    double rc2, int32_t* __restrict__ newpos, int32_t* __restrict__ deg) {
  const int lane = threadIdx.x & 31;
  const int64_t l = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (l >= n) return;
  const int64_t ai = aid[l];
  const double xi = pos[3 * ai], yi = pos[3 * ai + 1], zi = pos[3 * ai + 2];
  int count = 0;
  for (int b = c_rowptr[l]; b < c_rowptr[l + 1]; b += 32) {
    const int e = b + lane;
    bool ok = false;
    if (e < c_rowptr[l + 1]) {
      const int64_t aj = aid[c_send[e]];
      const uint32_t ps = (uint32_t)c_shift[e];
      double rx, ry, rz;
      const double d2 = canonical_rvec(cell.c, (int)((ps >> 16) & 255) - 128, (int)((ps >> 8) & 255) - 128, (int)(ps & 255) - 128, xi,
                                       yi, zi, pos[3 * aj], pos[3 * aj + 1], pos[3 * aj + 2], rx, ry, rz);
      ok = d2 < rc2;
    }
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    if (e < c_rowptr[l + 1]) newpos[e] = ok ? count + __popc(m & ((1u << lane) - 1u)) : -1;
    count += __popc(m);
  }
  if (lane == 0) deg[l] = count;
}

// pass 2: write the surviving edges (rows stay sorted by (sender, shift)); newpos becomes the absolute position
__global__ void __launch_bounds__(256) k_skin_fill(int64_t n, const int32_t* __restrict__ c_rowptr,
                                                   const int32_t* __restrict__ c_send, const int32_t* __restrict__ c_shift,
                                                   const int32_t* __restrict__ aid, const double* __restrict__ pos, Cell9 cell,
                                                   const int32_t* __restrict__ rowptr, int32_t* __restrict__ newpos,
                                                   int32_t* __restrict__ recv, int32_t* __restrict__ send,
                                                   float4* __restrict__ rvec, int32_t* __restrict__ cand) {
  const int lane = threadIdx.x & 31;
  const int64_t l = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (l >= n) return;
  const int64_t ai = aid[l];
  const double xi = pos[3 * ai], yi = pos[3 * ai + 1], zi = pos[3 * ai + 2];
  const int base = rowptr[l];
  for (int e = c_rowptr[l] + lane; e < c_rowptr[l + 1]; e += 32) {
    const int k = newpos[e];
    if (k < 0) continue;
    const int j = c_send[e];
    const int64_t aj = aid[j];
    const uint32_t ps = (uint32_t)c_shift[e];
    double rx, ry, rz;
    const double d2 = canonical_rvec(cell.c, (int)((ps >> 16) & 255) - 128, (int)((ps >> 8) & 255) - 128, (int)(ps & 255) - 128, xi, yi,
                                     zi, pos[3 * aj], pos[3 * aj + 1], pos[3 * aj + 2], rx, ry, rz);
    const int o = base + k;
    recv[o] = (int32_t)l; send[o] = j; cand[o] = e;
    rvec[o] = make_float4((float)rx, (float)ry, (float)rz, (float)sqrt(d2));
    newpos[e] = o;
  }
}

// pass 3: reverse index of the filtered list through the reverse index of the candidates (d2 of an edge and of its
// reverse are the same floating-point number, so both survive or neither does)
__global__ void k_skin_rev(const int32_t* __restrict__ E_dyn, const int32_t* __restrict__ cand, const int32_t* __restrict__ c_rev,
                           const int32_t* __restrict__ newpos, int32_t* __restrict__ rev, int* __restrict__ status) {
  const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= *E_dyn) return;
  int r = newpos[c_rev[cand[o]]];
  if (r < 0) { atomicOr(status, MLIP_DEV_REV_MISSING); r = (int)o; }
  rev[o] = r;
}

// flag[0] = 1 when an atom is farther than sqrt(thr2) from where it was at the last rebuild
__global__ void k_skin_moved(int64_t N, const double* __restrict__ pos, const double* __restrict__ pos0, double thr2,
                             int* __restrict__ flag) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool far = false;
  if (i < N) {
    const double dx = pos[3 * i] - pos0[3 * i], dy = pos[3 * i + 1] - pos0[3 * i + 1], dz = pos[3 * i + 2] - pos0[3 * i + 2];
    far = dx * dx + dy * dy + dz * dz > thr2;
  }
  if (__any_sync(0xffffffffu, far) && (threadIdx.x & 31) == 0) atomicOr(flag, 1);
}
}  // namespace

void SkinSub::release(mlip_ctx* ctx) {
  ctx->free(aid); ctx->free(c_shift); ctx->free(rowptr); ctx->free(recv); ctx->free(send); ctx->free(rev); ctx->free(rvec);
  ctx->free(newpos); ctx->free(cand); ctx->free(deg);
  aid = c_shift = rowptr = recv = send = rev = newpos = cand = deg = nullptr;
  rvec = nullptr;
}

int mlip_skin_sub_create(mlip_ctx* ctx, const mlip_graph* G, const PartSub* S, SkinSub* out) {
  cudaStream_t st = ctx->stream;
  const SubGraph c = S ? S->g : G->view();
  SkinSub& k = *out;
  k.n = c.n; k.E_cap = c.E;
  k.c_rowptr = c.rowptr; k.c_send = c.send; k.c_rev = c.rev;
  MLIP_TRY(ctx->alloc(&k.aid, c.n)); MLIP_TRY(ctx->alloc(&k.c_shift, c.E));
  MLIP_TRY(ctx->alloc(&k.rowptr, c.n + 1)); MLIP_TRY(ctx->alloc(&k.recv, c.E)); MLIP_TRY(ctx->alloc(&k.send, c.E));
  MLIP_TRY(ctx->alloc(&k.rev, c.E)); MLIP_TRY(ctx->alloc(&k.rvec, c.E)); MLIP_TRY(ctx->alloc(&k.newpos, c.E));
  MLIP_TRY(ctx->alloc(&k.cand, c.E)); MLIP_TRY(ctx->alloc(&k.deg, c.n + 1));
  const int64_t m = c.n > c.E ? c.n : c.E;
  if (m > 0) {
    k_skin_gather_sub<<<nblk(m, 256), 256, 0, st>>>(c.n, c.E, S ? S->gid : nullptr, G->perm, S ? S->geid : nullptr, G->shift, k.aid,
                                                    k.c_shift);
    ctx->launches++;
  }
  // the view the model kernels get: same atoms, classes and capacities as the candidate sub-graph, filtered edge arrays,
  // forces and per-atom energies scattered straight to the caller's numbering
  k.g = c;
  k.g.dyn = true;
  k.g.gid = k.aid;
  k.g.rowptr = k.rowptr; k.g.recv = k.recv; k.g.send = k.send; k.g.rev = k.rev; k.g.rvec = k.rvec;
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}

int mlip_skin_filter(mlip_ctx* ctx, const SkinSub& k, const double* pos_dev, const double* cell_host, double r_cut) {
  if (k.n == 0) return MLIP_OK;
  cudaStream_t st = ctx->stream;
  Cell9 cell;
  for (int i = 0; i < 9; ++i) cell.c[i] = cell_host[i];
  k_skin_count<<<nblk(k.n * 32, 256), 256, 0, st>>>(k.n, k.c_rowptr, k.c_send, k.c_shift, k.aid, pos_dev, cell, r_cut * r_cut, k.newpos,
                                                    k.deg);
  ctx->launches++;
  MLIP_TRY(mlip_exclusive_scan_i32(ctx, k.deg, k.rowptr, k.n, nullptr));
  k_skin_fill<<<nblk(k.n * 32, 256), 256, 0, st>>>(k.n, k.c_rowptr, k.c_send, k.c_shift, k.aid, pos_dev, cell, k.rowptr, k.newpos, k.recv,
                                                   k.send, k.rvec, k.cand);
  ctx->launches++;
  if (k.E_cap > 0) {
    k_skin_rev<<<nblk(k.E_cap, 256), 256, 0, st>>>(k.rowptr + k.n, k.cand, k.c_rev, k.newpos, k.rev, ctx->dev_status);
    ctx->launches++;
  }
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}

int mlip_skin_moved(mlip_ctx* ctx, int64_t N, const double* pos_dev, const double* pos0_dev, double skin, int* flag_dev) {
  cudaMemsetAsync(flag_dev, 0, sizeof(int), ctx->stream);
  if (N > 0) {
    k_skin_moved<<<nblk(N, 256), 256, 0, ctx->stream>>>(N, pos_dev, pos0_dev, 0.25 * skin * skin, flag_dev);
    ctx->launches++;
  }
  return MLIP_OK;
}
