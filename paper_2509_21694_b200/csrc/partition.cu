// Spatial partition + halo (PAPER.md:157 Stage 1, PAPER.md:165 Stage 2 with the geometric halo of
// reading R2) and construction of each extended sub-graph as the sub-graph of the global graph
// induced on the extended atom set (O6). Step A5 of SURVEY.md 8(a). Integer work + float64
// comparisons on fractional coordinates.
#include <math.h>
#include "common.cuh"

namespace {
struct BinGeom {
  int grid[3];
  int bin[3];
  double halo_frac[3];      // halo / perpendicular width
  double width_over_rc[3];  // perpendicular width / r_cut: fractional distance -> distance in units of r_c
};

// Depth class of every atom for one bin. Geometric rule: 0 = root (owned), k >= 1 = halo atom whose largest per-axis
// periodic distance to the bin lies in ((k-1) r_c, k r_c] (clamped to n_cls-1), -1 = outside the extended box. The 1e-9
// slack only ever moves an atom to a LOWER class (more work, never a missing term). With bfs != 0 the halo atoms are
// only marked CLS_UNSET here and get their class from the breadth-first search below.
constexpr int CLS_UNSET = 1 << 20;
__global__ void k_part_flags(int64_t N, const double* __restrict__ frac, BinGeom b, int n_cls, int bfs,
                             int32_t* __restrict__ cls) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  bool own = true, in_ext = true;
  int depth = 0;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double f = frac[3 * i + k];
    int bin = (int)floor(f * b.grid[k]);
    if (bin > b.grid[k] - 1) bin = b.grid[k] - 1;
    own = own && (bin == b.bin[k]);
    const double lo = (double)b.bin[k] / b.grid[k], hi = (double)(b.bin[k] + 1) / b.grid[k];
    double dist = 0.0;
    if (!(f >= lo && f < hi)) {
      double below = lo - f; below -= floor(below);
      double above = f - hi; above -= floor(above);
      dist = below < above ? below : above;
    }
    in_ext = in_ext && (dist <= b.halo_frac[k]);
    const int dk = (int)ceil(dist * b.width_over_rc[k] - 1e-9);
    depth = dk > depth ? dk : depth;
  }
  int c = -1;
  if (own) c = 0;
  else if (in_ext) c = bfs ? CLS_UNSET : (depth < 1 ? 1 : (depth > n_cls - 1 ? n_cls - 1 : depth));
  cls[i] = c;
}

// One level of the K-hop search of PAPER.md:165 (Stage 2), pull form: an unreached atom of the extended box takes
// class k if one of its neighbours has class k-1. The radius graph is symmetric, so the senders of the in-edges of i
// are its neighbours. Writes (k) never collide with the value tested (k-1): in place, no atomics, deterministic.
__global__ void __launch_bounds__(256) k_part_bfs(int64_t N, int k, const int32_t* __restrict__ rowptr,
                                                  const int32_t* __restrict__ send, int32_t* __restrict__ cls) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N || cls[i] != CLS_UNSET) return;
  for (int e = rowptr[i]; e < rowptr[i + 1]; ++e)
    if (cls[send[e]] == k - 1) { cls[i] = k; return; }
}

// flag of atom i in the class-major array ext[class * N + i], so that ONE exclusive scan over n_cls * N entries numbers
// the extended atoms by (class, cell order); atoms the search did not reach within n_cls-1 hops leave the sub-domain
__global__ void k_part_mark(int64_t N, int n_cls, int32_t* __restrict__ cls, int32_t* __restrict__ ext) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  int c = cls[i];
  if (c >= n_cls) { c = -1; cls[i] = -1; }
  if (c >= 0) ext[(int64_t)c * N + i] = 1;
}

__global__ void k_part_compact(int64_t N, const int32_t* __restrict__ cls, const int32_t* __restrict__ scan,
                               const int32_t* __restrict__ species, int32_t* __restrict__ lid,
                               int32_t* __restrict__ gid, float* __restrict__ omega, int32_t* __restrict__ species_l) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int c = cls[i];
  if (c >= 0) {
    const int l = scan[(int64_t)c * N + i];
    lid[i] = l;
    gid[l] = (int32_t)i;
    omega[l] = c == 0 ? 1.0f : 0.0f;
    species_l[l] = species[i];
  } else {
    lid[i] = -1;
  }
}

template <bool FILL>
__global__ void __launch_bounds__(256) k_part_edges(int64_t n_ext, const int32_t* __restrict__ gid,
                                                    const int32_t* __restrict__ lid,
                                                    const int32_t* __restrict__ g_rowptr,
                                                    const int32_t* __restrict__ g_send,
                                                    const float4* __restrict__ g_rvec, int32_t* __restrict__ deg,
                                                    const int32_t* __restrict__ rowptr, int32_t* __restrict__ recv,
                                                    int32_t* __restrict__ send, float4* __restrict__ rvec,
                                                    int32_t* __restrict__ geid) {
  const int lane = threadIdx.x & 31;
  const int64_t l = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (l >= n_ext) return;
  const int i = gid[l];
  const int lo = g_rowptr[i], hi = g_rowptr[i + 1];
  int count = 0;
  const int base = FILL ? rowptr[l] : 0;
  for (int b = lo; b < hi; b += 32) {
    const int e = b + lane;
    int sl = -1;
    if (e < hi) sl = lid[g_send[e]];
    const unsigned m = __ballot_sync(0xffffffffu, sl >= 0);
    if (FILL && sl >= 0) {
      const int o = base + count + __popc(m & ((1u << lane) - 1u));
      recv[o] = (int32_t)l;
      send[o] = sl;
      rvec[o] = g_rvec[e];
      geid[o] = e;
    }
    count += __popc(m);
  }
  if (!FILL && lane == 0) deg[l] = count;
}

__global__ void k_part_rev(int64_t E, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ send,
                           const int32_t* __restrict__ geid, const int32_t* __restrict__ g_rev,
                           int32_t* __restrict__ rev, int* __restrict__ err_flag) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= E) return;
  const int want = g_rev[geid[e]];
  const int j = send[e];
  int lo = rowptr[j], hi = rowptr[j + 1] - 1, found = -1;
  while (lo <= hi) {
    const int mid = (lo + hi) >> 1;
    const int v = geid[mid];
    if (v == want) { found = mid; break; }
    if (v < want) lo = mid + 1; else hi = mid - 1;
  }
  if (found < 0) *err_flag = 3;
  rev[e] = found;
}

inline unsigned nblk(int64_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }

void free_sub(mlip_ctx* c, PartSub& s) {
  c->free(s.gid); c->free(s.species); c->free(s.rowptr); c->free(s.recv); c->free(s.send); c->free(s.rev);
  c->free(s.omega); c->free(s.rvec); c->free(s.geid);
}
}  // namespace

extern "C" void mlip_part_destroy(mlip_part* p) {
  if (!p) return;
  for (auto& s : p->subs) free_sub(p->ctx, s);
  delete p;
}

extern "C" int mlip_partition_grid(mlip_ctx* ctx, const mlip_graph* G, const int grid[3], double halo,
                                   mlip_part** out) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!G) { ctx->set_error("mlip_partition_grid: invalid argument"); return MLIP_ERR_INVALID_ARG; }
  return mlip_partition_grid_ex(ctx, G, grid, halo, halo, G->r_cut, false, false, out);
}

// halo_box: width of the geometric box the extended set is searched in; halo / r_class: the number of shells
// K = ceil(halo / r_class) (depth classes, levels of the K-hop search). The public call uses halo_box = halo and
// r_class = the graph's cutoff; the Verlet-skin MD driver partitions the CANDIDATE graph (cutoff r_c + skin) with
// halo_box = halo + skin (atoms move by up to skin/2 each before the next rebuild) and r_class = r_c, forces the K-hop
// rule (hop counts over the candidate graph are lower bounds of the hop counts over any later exact graph) and keeps the
// global edge id of every sub-domain edge.
int mlip_partition_grid_ex(mlip_ctx* ctx, const mlip_graph* G, const int grid[3], double halo_box, double halo,
                           double r_class, bool force_khop, bool keep_geid, mlip_part** out, int shard, int n_shards) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (n_shards < 1 || shard < 0 || shard >= n_shards) { ctx->set_error("mlip_partition_grid_shard: shard outside [0, n_shards)"); return MLIP_ERR_INVALID_ARG; }
  if (!G || !grid || !out || grid[0] < 1 || grid[1] < 1 || grid[2] < 1 || !(halo >= 0.0) || !(halo_box >= halo) || !(r_class > 0.0)) {
    ctx->set_error("mlip_partition_grid: invalid argument");
    return MLIP_ERR_INVALID_ARG;
  }
  *out = nullptr;
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  const int64_t N = G->N;
  mlip_part* P = new mlip_part();
  P->ctx = ctx; P->halo = halo; P->N = N; P->shard = shard; P->n_shards = n_shards;
  for (int k = 0; k < 3; ++k) P->grid[k] = grid[k];
  auto fail = [&](int code) { mlip_part_destroy(P); return code; };
  ProfScope prof(ctx, MLIP_PROF_PARTITION);
#define P_TRY(x) do { int _s = (x); if (_s != MLIP_OK) return fail(_s); } while (0)
  // depth classes 0 .. n_cls-1 (see SubGraph): the halo spans ceil(halo / r_c) shells of thickness r_c
  int n_cls = 1 + (int)ceil(halo / r_class - 1e-9);
  if (n_cls < 2) n_cls = 2;
  if (n_cls > MLIP_MAX_CLS) {
    ctx->set_error("partition: halo spans more than 31 shells of thickness r_cut (ceil(halo / r_cut) > 31)");
    return fail(MLIP_ERR_UNSUPPORTED);
  }
  const bool bfs = ctx->khop_halo || force_khop;
  P->khop = bfs;
  const int64_t CN = (int64_t)n_cls * N;
  if (CN >= (int64_t)1 << 31) { ctx->set_error("partition: n_cls * N >= 2^31"); return fail(MLIP_ERR_OVERFLOW); }
  int32_t *ext = nullptr, *cls = nullptr, *scan = nullptr, *lid = nullptr, *deg = nullptr, *geid = nullptr;
  int* err_flag = nullptr;
  P_TRY(ctx->alloc(&ext, CN + 1)); P_TRY(ctx->alloc(&cls, N + 1)); P_TRY(ctx->alloc(&scan, CN + 1));
  P_TRY(ctx->alloc(&lid, N + 1)); P_TRY(ctx->alloc(&err_flag, 1));
  cudaMemsetAsync(err_flag, 0, sizeof(int), st);
  for (int bx = 0; bx < grid[0]; ++bx)
    for (int by = 0; by < grid[1]; ++by)
      for (int bz = 0; bz < grid[2]; ++bz) {
        BinGeom b;
        b.bin[0] = bx; b.bin[1] = by; b.bin[2] = bz;
        for (int k = 0; k < 3; ++k) {
          b.grid[k] = grid[k]; b.halo_frac[k] = halo_box / G->width[k]; b.width_over_rc[k] = G->width[k] / r_class;
        }
        P->subs.emplace_back();
        PartSub& S = P->subs.back();
        // sub-domains of other shards stay empty handles: their place in the numbering k = (bx, by, bz) is kept
        if ((int)((P->subs.size() - 1) % (size_t)n_shards) != shard) continue;
        int64_t n_ext = 0, E = 0;
        int32_t cls_start[MLIP_MAX_CLS + 1] = {0}, E_at[MLIP_MAX_CLS] = {0};
        cudaMemsetAsync(ext, 0, sizeof(int32_t) * (CN + 1), st);
        if (N > 0) {
          k_part_flags<<<nblk(N, 256), 256, 0, st>>>(N, G->frac, b, n_cls, bfs ? 1 : 0, cls);
          ctx->launches++;
          for (int k = 1; bfs && k < n_cls; ++k) {
            k_part_bfs<<<nblk(N, 256), 256, 0, st>>>(N, k, G->rowptr, G->send, cls);
            ctx->launches++;
          }
          k_part_mark<<<nblk(N, 256), 256, 0, st>>>(N, n_cls, cls, ext);
          ctx->launches++;
        }
        P_TRY(mlip_exclusive_scan_i32(ctx, ext, scan, CN, nullptr));
        // first local id of every class (scan[c * N]) and the total (scan[n_cls * N])
        for (int c = 0; c <= n_cls && N > 0; ++c)
          cudaMemcpyAsync(&cls_start[c], scan + (int64_t)c * N, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        if (cudaStreamSynchronize(st) != cudaSuccess) { ctx->set_error("partition: scan failed"); return fail(MLIP_ERR_CUDA); }
        n_ext = N > 0 ? cls_start[n_cls] : 0;
        P_TRY(ctx->alloc(&S.gid, n_ext)); P_TRY(ctx->alloc(&S.omega, n_ext)); P_TRY(ctx->alloc(&S.species, n_ext));
        P_TRY(ctx->alloc(&S.rowptr, n_ext + 1)); P_TRY(ctx->alloc(&deg, n_ext + 1));
        if (N > 0) {
          k_part_compact<<<nblk(N, 256), 256, 0, st>>>(N, cls, scan, G->species, lid, S.gid, S.omega, S.species);
          ctx->launches++;
        }
        if (n_ext > 0) {
          k_part_edges<false><<<nblk(n_ext * 32, 256), 256, 0, st>>>(n_ext, S.gid, lid, G->rowptr, G->send, G->rvec,
                                                                     deg, nullptr, nullptr, nullptr, nullptr, nullptr);
          ctx->launches++;
        }
        P_TRY(mlip_exclusive_scan_i32(ctx, deg, S.rowptr, n_ext, nullptr));
        // E_le[c] = rowptr[n_le[c]], n_le[c] = first local id of class c+1
        for (int c = 0; c < n_cls; ++c)
          cudaMemcpyAsync(&E_at[c], S.rowptr + (N > 0 ? cls_start[c + 1] : 0), sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        if (cudaStreamSynchronize(st) != cudaSuccess) { ctx->set_error("partition: scan failed"); return fail(MLIP_ERR_CUDA); }
        E = E_at[n_cls - 1];
        P_TRY(ctx->alloc(&S.recv, E)); P_TRY(ctx->alloc(&S.send, E)); P_TRY(ctx->alloc(&S.rev, E));
        P_TRY(ctx->alloc(&S.rvec, E)); P_TRY(ctx->alloc(&geid, E));
        if (E > 0) {
          k_part_edges<true><<<nblk(n_ext * 32, 256), 256, 0, st>>>(n_ext, S.gid, lid, G->rowptr, G->send, G->rvec,
                                                                    nullptr, S.rowptr, S.recv, S.send, S.rvec, geid);
          k_part_rev<<<nblk(E, 256), 256, 0, st>>>(E, S.rowptr, S.send, geid, G->rev, S.rev, err_flag);
          ctx->launches += 2;
        }
        ctx->free(deg); deg = nullptr;
        if (keep_geid) S.geid = geid; else ctx->free(geid);
        geid = nullptr;
        S.g.n = n_ext; S.g.n_owned = N > 0 ? cls_start[1] : 0; S.g.E = E;
        S.g.n_cls = n_cls;
        for (int c = 0; c < n_cls; ++c) { S.g.n_le[c] = N > 0 ? cls_start[c + 1] : 0; S.g.E_le[c] = E_at[c]; }
        S.g.gid = S.gid; S.g.omega = S.omega; S.g.species = S.species; S.g.rowptr = S.rowptr;
        S.g.recv = S.recv; S.g.send = S.send; S.g.rev = S.rev; S.g.rvec = S.rvec;
      }
  int err_h = 0;
  cudaMemcpyAsync(&err_h, err_flag, sizeof(int), cudaMemcpyDeviceToHost, st);
  cudaError_t e = cudaStreamSynchronize(st);
  ctx->free(ext); ctx->free(cls); ctx->free(scan); ctx->free(lid); ctx->free(err_flag);
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) {
    ctx->set_error(std::string("partition: ") + cudaGetErrorString(e));
    return fail(MLIP_ERR_CUDA);
  }
  if (err_h != 0) { ctx->set_error("partition: reverse edge not found (internal error)"); return fail(MLIP_ERR_CUDA); }
#undef P_TRY
  *out = P;
  return MLIP_OK;
}

extern "C" int mlip_partition_grid_shard(mlip_ctx* ctx, const mlip_graph* G, const int grid[3], double halo, int shard,
                                         int n_shards, mlip_part** out) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!G) { ctx->set_error("mlip_partition_grid_shard: invalid argument"); return MLIP_ERR_INVALID_ARG; }
  return mlip_partition_grid_ex(ctx, G, grid, halo, halo, G->r_cut, false, false, out, shard, n_shards);
}

extern "C" int mlip_partition(mlip_ctx* ctx, const mlip_graph* G, int n_sub, double halo, mlip_part** out) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!G || n_sub < 1) { ctx->set_error("mlip_partition: invalid argument"); return MLIP_ERR_INVALID_ARG; }
  int axis = 0;
  for (int k = 1; k < 3; ++k) if (G->width[k] > G->width[axis]) axis = k;  // ties -> lowest index (R3)
  int grid[3] = {1, 1, 1};
  grid[axis] = n_sub;
  return mlip_partition_grid(ctx, G, grid, halo, out);
}

extern "C" int mlip_part_count(const mlip_part* p, int* n_sub) {
  if (!p || !n_sub) return MLIP_ERR_INVALID_ARG;
  *n_sub = (int)p->subs.size();
  return MLIP_OK;
}

extern "C" int mlip_part_info(const mlip_part* p, int s, int64_t* n_owned, int64_t* n_ext, int64_t* n_edges) {
  if (!p || s < 0 || s >= (int)p->subs.size()) return MLIP_ERR_INVALID_ARG;
  if (n_owned) *n_owned = p->subs[s].g.n_owned;
  if (n_ext) *n_ext = p->subs[s].g.n;
  if (n_edges) *n_edges = p->subs[s].g.E;
  return MLIP_OK;
}

extern "C" int mlip_part_layer_info(const mlip_part* p, int s, int L, int l, int64_t* n_recv, int64_t* n_send,
                                    int64_t* n_edges) {
  if (!p || s < 0 || s >= (int)p->subs.size() || L < 1 || l < 0 || l >= L) return MLIP_ERR_INVALID_ARG;
  const SubGraph& g = p->subs[s].g;
  const bool act = p->ctx->active_sets;
  if (n_recv) *n_recv = act ? g.atoms_upto(L - 1 - l) : g.n;
  if (n_send) *n_send = act ? g.atoms_upto(L - l) : g.n;
  if (n_edges) *n_edges = act ? g.edges_upto(L - 1 - l) : g.E;
  return MLIP_OK;
}
