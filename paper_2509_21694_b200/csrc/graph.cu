// Radius graph under periodic boundaries by a cell list: counting sort of atoms
// by cell id + prefix sums, stencil traversal with explicit image shifts, canonical float64
// accept predicate (reading R10: fixed operation order, no FMA contraction), per-row sort by
// (sender, shift), reverse-edge index. Steps A1-A4 of SURVEY.md 8(a).
#include <math.h>
#include <string.h>
#include "canon.cuh"
#include "common.cuh"

namespace {

struct CellGeom {
  double cell[9];  // rows a1,a2,a3
  double inv[9];   // inverse, frac = pos . inv
  double rc2;
  int nc[3];
  int R[3];
};

__device__ __forceinline__ int floordiv(int a, int b) { int q = a / b; return (a % b != 0 && ((a < 0) != (b < 0))) ? q - 1 : q; }

// ---- A1: fractional coordinates, wrap counts, cell id, cell histogram ------------------------
__global__ void k_frac_bin(const double* __restrict__ pos, int64_t N, CellGeom g,
                           double* __restrict__ frac, int32_t* __restrict__ wrap,
                           int32_t* __restrict__ cellid, int32_t* __restrict__ cell_count) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
  int c[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    double f = x * g.inv[0 + k] + y * g.inv[3 + k] + z * g.inv[6 + k];
    double w = floor(f);
    double fw = f - w;
    if (fw >= 1.0) { fw = 0.0; w += 1.0; }
    frac[3 * i + k] = fw;
    wrap[3 * i + k] = (int32_t)w;
    int ck = (int)(fw * g.nc[k]);
    c[k] = ck >= g.nc[k] ? g.nc[k] - 1 : ck;
  }
  const int id = (c[0] * g.nc[1] + c[1]) * g.nc[2] + c[2];
  cellid[i] = id;
  atomicAdd(&cell_count[id], 1);
}

// ---- A2: counting-sort scatter, then order each cell by atom index (deterministic) -----------
__global__ void k_cell_scatter(const int32_t* __restrict__ cellid, int64_t N,
                               const int32_t* __restrict__ cell_start, int32_t* __restrict__ cursor,
                               int32_t* __restrict__ order) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int c = cellid[i];
  order[cell_start[c] + atomicAdd(&cursor[c], 1)] = (int32_t)i;
}

__global__ void k_cell_sort(const int32_t* __restrict__ cell_start, int n_cells, int32_t* __restrict__ order) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cells) return;
  const int lo = cell_start[c], hi = cell_start[c + 1];
  for (int a = lo + 1; a < hi; ++a) {  // insertion sort, cells hold O(10) atoms
    int v = order[a], b = a - 1;
    while (b >= lo && order[b] > v) { order[b + 1] = order[b]; --b; }
    order[b + 1] = v;
  }
}

__global__ void k_gather_sorted(const int32_t* __restrict__ order, int64_t N,
                                const double* __restrict__ pos, const double* __restrict__ frac,
                                const int32_t* __restrict__ wrap, const int32_t* __restrict__ species,
                                const int32_t* __restrict__ cellid,
                                double* __restrict__ pos_s, double* __restrict__ frac_s,
                                int32_t* __restrict__ wrap_s, int32_t* __restrict__ species_s,
                                int32_t* __restrict__ cellid_s, int* __restrict__ sp_range /*[2]: max(s), max(-s)*/) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int sp = k < N ? species[order[k]] : 0;
  const int hi = __reduce_max_sync(0xffffffffu, sp), lo = __reduce_max_sync(0xffffffffu, -sp);
  if ((threadIdx.x & 31) == 0) {
    if (hi > 0) atomicMax(&sp_range[0], hi);
    if (lo > 0) atomicMax(&sp_range[1], lo);
  }
  if (k >= N) return;
  const int64_t i = order[k];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    pos_s[3 * k + a] = pos[3 * i + a];
    frac_s[3 * k + a] = frac[3 * i + a];
    wrap_s[3 * k + a] = wrap[3 * i + a];
  }
  species_s[k] = species[i];
  cellid_s[k] = cellid[i];
}

// ---- A3: stencil traversal --------------------------------------------------------------------
// One warp per atom. FILL=false counts accepted neighbours, FILL=true writes 64-bit keys
// (sender << 24 | packed shift) to the row in traversal order (sorted afterwards).
__device__ __forceinline__ uint32_t pack_shift(int nx, int ny, int nz) {
  return ((uint32_t)(nx + 128) << 16) | ((uint32_t)(ny + 128) << 8) | (uint32_t)(nz + 128);
}

// MODE 0: count. MODE 1: fill the CSR rows (base = rowptr[i]). MODE 2: count AND write the keys of atom i to the
// fixed-capacity row [i * cap, (i + 1) * cap) of a scratch buffer, so that the 27-cell search runs once; a row that
// would overflow raises err_flag = 4 and the caller falls back to MODE 0 + MODE 1.
template <int MODE>
__global__ void __launch_bounds__(256) k_neighbors(int64_t N, CellGeom g,
                                                   const double* __restrict__ pos_s,
                                                   const int32_t* __restrict__ wrap_s,
                                                   const int32_t* __restrict__ cellid_s,
                                                   const int32_t* __restrict__ cell_start,
                                                   int32_t* __restrict__ deg,
                                                   const int32_t* __restrict__ rowptr,
                                                   unsigned long long* __restrict__ keys,
                                                   unsigned long long* __restrict__ total,
                                                   int* __restrict__ err_flag, int cap) {
  constexpr bool FILL = MODE != 0;
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  const double xi = pos_s[3 * i], yi = pos_s[3 * i + 1], zi = pos_s[3 * i + 2];
  const int wi0 = wrap_s[3 * i], wi1 = wrap_s[3 * i + 1], wi2 = wrap_s[3 * i + 2];
  const int id = cellid_s[i];
  const int c2 = id % g.nc[2];
  const int c1 = (id / g.nc[2]) % g.nc[1];
  const int c0 = id / (g.nc[2] * g.nc[1]);
  int count = 0;
  int64_t base = MODE == 1 ? (int64_t)rowptr[i] : (MODE == 2 ? i * (int64_t)cap : 0);
  for (int o0 = -g.R[0]; o0 <= g.R[0]; ++o0) {
    const int t0 = c0 + o0, s0 = floordiv(t0, g.nc[0]), cc0 = t0 - s0 * g.nc[0];
    for (int o1 = -g.R[1]; o1 <= g.R[1]; ++o1) {
      const int t1 = c1 + o1, s1 = floordiv(t1, g.nc[1]), cc1 = t1 - s1 * g.nc[1];
      const int rowbase = (cc0 * g.nc[1] + cc1) * g.nc[2];
      // cells along the fastest axis are contiguous in the sorted order: merge runs that share
      // the same image shift
      int o2 = -g.R[2];
      while (o2 <= g.R[2]) {
        const int t2 = c2 + o2, s2 = floordiv(t2, g.nc[2]), cc2 = t2 - s2 * g.nc[2];
        int run = 1;  // extend while the next cell is the next index with the same shift
        while (o2 + run <= g.R[2] && cc2 + run < g.nc[2]) ++run;
        const int lo = cell_start[rowbase + cc2], hi = cell_start[rowbase + cc2 + run];
        for (int b = lo; b < hi; b += 32) {
          const int j = b + lane;
          bool ok = false;
          uint32_t ps = 0;
          if (j < hi) {
            const int nx = s0 - wrap_s[3 * j] + wi0;
            const int ny = s1 - wrap_s[3 * j + 1] + wi1;
            const int nz = s2 - wrap_s[3 * j + 2] + wi2;
            // canonical predicate (O1): t = (nx*a1 + ny*a2) + nz*a3; r = (xj - xi) + t   (canon.cuh)
            double rx, ry, rz;
            const double d2 = canonical_rvec(g.cell, nx, ny, nz, xi, yi, zi, pos_s[3 * j], pos_s[3 * j + 1], pos_s[3 * j + 2], rx, ry, rz);
            ok = d2 < g.rc2 && !(j == i && nx == 0 && ny == 0 && nz == 0);
            if (ok && (nx < -127 || nx > 127 || ny < -127 || ny > 127 || nz < -127 || nz > 127)) {
              atomicOr(err_flag, 1);
              ok = false;
            }
            ps = pack_shift(nx, ny, nz);
          }
          const unsigned m = __ballot_sync(0xffffffffu, ok);
          if (FILL && ok) {
            const int rank = __popc(m & ((1u << lane) - 1u));
            if (MODE == 1 || count + rank < cap) keys[base + count + rank] = ((unsigned long long)(uint32_t)j << 24) | ps;
          }
          count += __popc(m);
        }
        o2 += run;
      }
    }
  }
  if (MODE != 1 && lane == 0) {
    deg[i] = count;
    atomicAdd(total, (unsigned long long)count);
    if (MODE == 2 && count > cap) atomicOr(err_flag, 4);
  }
}

// scratch rows of MODE 2 -> CSR rows
__global__ void __launch_bounds__(256) k_compact_keys(int64_t N, int cap, const int32_t* __restrict__ rowptr,
                                                      const unsigned long long* __restrict__ scratch,
                                                      unsigned long long* __restrict__ keys) {
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  const int lo = rowptr[i], len = rowptr[i + 1] - lo;
  for (int t = lane; t < len; t += 32) keys[lo + t] = scratch[i * (int64_t)cap + t];
}

// ---- per-row sort of 64-bit keys (one warp per row, bitonic in shared memory) ------------------
constexpr int SORT_MAX = 512;
__global__ void __launch_bounds__(128) k_sort_rows(int64_t n_rows, const int32_t* __restrict__ rowptr,
                                                   unsigned long long* __restrict__ keys) {
  __shared__ unsigned long long buf[4][SORT_MAX];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t row = (int64_t)blockIdx.x * 4 + w;
  if (row >= n_rows) return;
  const int lo = rowptr[row], len = rowptr[row + 1] - lo;
  if (len <= 1) return;
  if (len > SORT_MAX) {  // very dense rows: slow but correct
    if (lane == 0) {
      for (int a = 1; a < len; ++a) {
        unsigned long long v = keys[lo + a];
        int b = a - 1;
        while (b >= 0 && keys[lo + b] > v) { keys[lo + b + 1] = keys[lo + b]; --b; }
        keys[lo + b + 1] = v;
      }
    }
    return;
  }
  int P = 32;
  while (P < len) P <<= 1;
  for (int t = lane; t < P; t += 32) buf[w][t] = t < len ? keys[lo + t] : ~0ull;
  __syncwarp();
  for (int k = 2; k <= P; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int t = lane; t < P; t += 32) {
        const int p = t ^ j;
        if (p > t) {
          const unsigned long long a = buf[w][t], b = buf[w][p];
          const bool up = (t & k) == 0;
          if ((a > b) == up) { buf[w][t] = b; buf[w][p] = a; }
        }
      }
      __syncwarp();
    }
  }
  for (int t = lane; t < len; t += 32) keys[lo + t] = buf[w][t];
}

// ---- decode keys -> recv/send/shift/rvec (float64 difference, then rounded to fp32) ------------
__global__ void __launch_bounds__(256) k_finalize_edges(int64_t N, CellGeom g,
                                                        const double* __restrict__ pos_s,
                                                        const int32_t* __restrict__ rowptr,
                                                        const unsigned long long* __restrict__ keys,
                                                        int32_t* __restrict__ recv, int32_t* __restrict__ send,
                                                        int32_t* __restrict__ shift, float4* __restrict__ rvec) {
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  const double xi = pos_s[3 * i], yi = pos_s[3 * i + 1], zi = pos_s[3 * i + 2];
  const int lo = rowptr[i], hi = rowptr[i + 1];
  for (int e = lo + lane; e < hi; e += 32) {
    const unsigned long long k = keys[e];
    const int j = (int)(k >> 24);
    const uint32_t ps = (uint32_t)(k & 0xffffffu);
    double rx, ry, rz;
    const double d2 = canonical_rvec(g.cell, (int)((ps >> 16) & 255) - 128, (int)((ps >> 8) & 255) - 128, (int)(ps & 255) - 128, xi, yi, zi,
                                     pos_s[3 * j], pos_s[3 * j + 1], pos_s[3 * j + 2], rx, ry, rz);
    recv[e] = (int32_t)i;
    send[e] = j;
    shift[e] = (int32_t)ps;
    rvec[e] = make_float4((float)rx, (float)ry, (float)rz, (float)sqrt(d2));
  }
}

// ---- A4: reverse-edge index by binary search in the sender's row ------------------------------
__device__ __forceinline__ uint32_t negate_shift(uint32_t ps) {
  const int nx = (int)((ps >> 16) & 255) - 128, ny = (int)((ps >> 8) & 255) - 128, nz = (int)(ps & 255) - 128;
  return pack_shift(-nx, -ny, -nz);
}

__global__ void k_reverse(int64_t E, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ recv,
                          const unsigned long long* __restrict__ keys, int32_t* __restrict__ rev,
                          int* __restrict__ err_flag) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= E) return;
  const unsigned long long k = keys[e];
  const int j = (int)(k >> 24);
  const unsigned long long want = ((unsigned long long)(uint32_t)recv[e] << 24) | negate_shift((uint32_t)(k & 0xffffffu));
  int lo = rowptr[j], hi = rowptr[j + 1] - 1;
  int found = -1;
  while (lo <= hi) {
    const int mid = (lo + hi) >> 1;
    const unsigned long long v = keys[mid];
    if (v == want) { found = mid; break; }
    if (v < want) lo = mid + 1; else hi = mid - 1;
  }
  // a missing partner (impossible for a symmetric list) is reported through the context status word; the edge points
  // at itself so that nothing downstream indexes out of bounds
  if (found < 0) { atomicOr(err_flag, MLIP_DEV_REV_MISSING); found = (int)e; }
  rev[e] = found;
}

// ---- export in the caller's numbering, canonical order ----------------------------------------
__global__ void k_invert_perm(const int32_t* __restrict__ perm, int64_t N, int32_t* __restrict__ inv) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < N) inv[perm[k]] = (int32_t)k;
}
__global__ void k_export_deg(const int32_t* __restrict__ inv, const int32_t* __restrict__ rowptr, int64_t N,
                             int32_t* __restrict__ deg_orig) {
  const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a < N) { const int i = inv[a]; deg_orig[a] = rowptr[i + 1] - rowptr[i]; }
}
__global__ void __launch_bounds__(256) k_export_keys(int64_t N, const int32_t* __restrict__ inv,
                                                     const int32_t* __restrict__ perm,
                                                     const int32_t* __restrict__ rowptr,
                                                     const int32_t* __restrict__ send, const int32_t* __restrict__ shift,
                                                     const int32_t* __restrict__ rowptr_orig,
                                                     unsigned long long* __restrict__ keys) {
  const int lane = threadIdx.x & 31;
  const int64_t a = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= N) return;
  const int i = inv[a];
  const int lo = rowptr[i], len = rowptr[i + 1] - lo, out = rowptr_orig[a];
  for (int t = lane; t < len; t += 32)
    keys[out + t] = ((unsigned long long)(uint32_t)perm[send[lo + t]] << 24) | (uint32_t)shift[lo + t];
}
__global__ void __launch_bounds__(256) k_export_decode(int64_t N, const int32_t* __restrict__ rowptr_orig,
                                                       const unsigned long long* __restrict__ keys,
                                                       int32_t* __restrict__ recv, int32_t* __restrict__ send,
                                                       int32_t* __restrict__ shift3) {
  const int lane = threadIdx.x & 31;
  const int64_t a = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= N) return;
  for (int e = rowptr_orig[a] + lane; e < rowptr_orig[a + 1]; e += 32) {
    const unsigned long long k = keys[e];
    const uint32_t ps = (uint32_t)(k & 0xffffffu);
    recv[e] = (int32_t)a;
    send[e] = (int32_t)(k >> 24);
    shift3[3 * (int64_t)e + 0] = (int)((ps >> 16) & 255) - 128;
    shift3[3 * (int64_t)e + 1] = (int)((ps >> 8) & 255) - 128;
    shift3[3 * (int64_t)e + 2] = (int)(ps & 255) - 128;
  }
}

bool invert3(const double* m, double* inv, double* vol) {
  const double a = m[0], b = m[1], c = m[2], d = m[3], e = m[4], f = m[5], g = m[6], h = m[7], i = m[8];
  const double det = a * (e * i - f * h) - b * (d * i - f * g) + c * (d * h - e * g);
  *vol = fabs(det);
  if (!(fabs(det) > 1e-12)) return false;
  const double id = 1.0 / det;
  inv[0] = (e * i - f * h) * id; inv[1] = (c * h - b * i) * id; inv[2] = (b * f - c * e) * id;
  inv[3] = (f * g - d * i) * id; inv[4] = (a * i - c * g) * id; inv[5] = (c * d - a * f) * id;
  inv[6] = (d * h - e * g) * id; inv[7] = (b * g - a * h) * id; inv[8] = (a * e - b * d) * id;
  return true;
}
void cross3(const double* u, const double* v, double* o) {
  o[0] = u[1] * v[2] - u[2] * v[1]; o[1] = u[2] * v[0] - u[0] * v[2]; o[2] = u[0] * v[1] - u[1] * v[0];
}
double norm3(const double* u) { return sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]); }

inline unsigned nblk(int64_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }
}  // namespace

extern "C" int mlip_build_graph(mlip_ctx* ctx, const double* pos_dev, const double* cell_host,
                                const int32_t* species_dev, int64_t N, double r_cut, mlip_graph** out) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!out || !cell_host || N < 0 || (N > 0 && (!pos_dev || !species_dev)) || !(r_cut > 0)) {
    ctx->set_error("mlip_build_graph: invalid argument");
    return MLIP_ERR_INVALID_ARG;
  }
  *out = nullptr;
  if (N >= (int64_t)1 << 31) { ctx->set_error("too many atoms"); return MLIP_ERR_OVERFLOW; }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  CellGeom g;
  memcpy(g.cell, cell_host, sizeof(g.cell));
  double vol;
  if (!invert3(g.cell, g.inv, &vol)) { ctx->set_error("singular cell"); return MLIP_ERR_UNSUPPORTED; }
  double c12[3], c20[3], c01[3], width[3];
  cross3(g.cell + 3, g.cell + 6, c12); cross3(g.cell + 6, g.cell + 0, c20); cross3(g.cell + 0, g.cell + 3, c01);
  width[0] = vol / norm3(c12); width[1] = vol / norm3(c20); width[2] = vol / norm3(c01);
  int64_t n_cells = 1;
  for (int k = 0; k < 3; ++k) {
    const double rc = r_cut * (1.0 + 1e-6);  // slack so that binning round-off cannot lose a pair
    int nc = (int)floor(width[k] / rc);
    if (nc < 1) nc = 1;
    if (nc > 1024) nc = 1024;
    g.nc[k] = nc;
    g.R[k] = (int)ceil(rc / (width[k] / nc));
    n_cells *= nc;
  }
  // keep the cell table proportional to the atom count (sparse boxes): coarsen the finest axis
  while (n_cells > 8 * N + 4096) {
    int k = 0;
    for (int a = 1; a < 3; ++a) if (g.nc[a] > g.nc[k]) k = a;
    n_cells /= g.nc[k];
    g.nc[k] = (g.nc[k] + 1) / 2;
    g.R[k] = (int)ceil(r_cut * (1.0 + 1e-6) / (width[k] / g.nc[k]));
    n_cells *= g.nc[k];
  }
  g.rc2 = r_cut * r_cut;
  cudaStream_t st = ctx->stream;

  mlip_graph* G = new mlip_graph();
  G->ctx = ctx; G->N = N; G->r_cut = r_cut;
  memcpy(G->cell, g.cell, sizeof(g.cell)); memcpy(G->inv, g.inv, sizeof(g.inv));
  memcpy(G->width, width, sizeof(width)); memcpy(G->nc, g.nc, sizeof(g.nc));
  auto fail = [&](int code) { mlip_graph_destroy(G); return code; };
  ProfScope prof(ctx, MLIP_PROF_GRAPH);

  double *frac = nullptr, *pos_s = nullptr;
  int32_t *wrap = nullptr, *cellid = nullptr, *cell_count = nullptr, *cell_start = nullptr, *order = nullptr,
          *wrap_s = nullptr, *cellid_s = nullptr, *deg = nullptr;
  unsigned long long *keys = nullptr, *total = nullptr, *scratch = nullptr;
  int cap = 0;
  int *err_flag = nullptr, *sp_range = nullptr;
#define G_TRY(x) do { int _s = (x); if (_s != MLIP_OK) return fail(_s); } while (0)
  G_TRY(ctx->alloc(&frac, 3 * N)); G_TRY(ctx->alloc(&wrap, 3 * N)); G_TRY(ctx->alloc(&cellid, N));
  G_TRY(ctx->alloc(&cell_count, 2 * n_cells + 2)); G_TRY(ctx->alloc(&cell_start, n_cells + 1));
  G_TRY(ctx->alloc(&order, N)); G_TRY(ctx->alloc(&pos_s, 3 * N)); G_TRY(ctx->alloc(&wrap_s, 3 * N));
  G_TRY(ctx->alloc(&cellid_s, N)); G_TRY(ctx->alloc(&deg, N + 1)); G_TRY(ctx->alloc(&total, 2));
  G_TRY(ctx->alloc(&err_flag, 1)); G_TRY(ctx->alloc(&sp_range, 2));
  G_TRY(ctx->alloc(&G->perm, N)); G_TRY(ctx->alloc(&G->frac, 3 * N)); G_TRY(ctx->alloc(&G->species, N));
  G_TRY(ctx->alloc(&G->rowptr, N + 1));
  int32_t* cursor = cell_count + n_cells + 1;
  cudaMemsetAsync(cell_count, 0, sizeof(int32_t) * (2 * n_cells + 2), st);
  cudaMemsetAsync(total, 0, 2 * sizeof(unsigned long long), st);
  cudaMemsetAsync(err_flag, 0, sizeof(int), st);
  cudaMemsetAsync(sp_range, 0, 2 * sizeof(int), st);
  if (N > 0) {
    k_frac_bin<<<nblk(N, 256), 256, 0, st>>>(pos_dev, N, g, frac, wrap, cellid, cell_count);
    ctx->launches++;
  }
  G_TRY(mlip_exclusive_scan_i32(ctx, cell_count, cell_start, n_cells, nullptr));
  if (N > 0) {
    k_cell_scatter<<<nblk(N, 256), 256, 0, st>>>(cellid, N, cell_start, cursor, order);
    k_cell_sort<<<nblk(n_cells, 128), 128, 0, st>>>(cell_start, (int)n_cells, order);
    k_gather_sorted<<<nblk(N, 256), 256, 0, st>>>(order, N, pos_dev, frac, wrap, species_dev, cellid, pos_s,
                                                  G->frac, wrap_s, G->species, cellid_s, sp_range);
    cudaMemcpyAsync(G->perm, order, sizeof(int32_t) * N, cudaMemcpyDeviceToDevice, st);
    // one search pass when a capped scratch row per atom is affordable: cap = 1.5 x the mean degree + 32
    const double nbar = 4.18879020478639 * r_cut * r_cut * r_cut * (double)N / vol;
    cap = (int)(1.5 * nbar + 32.0);
    cap = (cap + 7) & ~7;
    if ((double)N * cap * 8.0 <= 2.0e9 && ctx->alloc(&scratch, (size_t)N * cap) == MLIP_OK) {
      k_neighbors<2><<<nblk(N * 32, 256), 256, 0, st>>>(N, g, pos_s, wrap_s, cellid_s, cell_start, deg, nullptr,
                                                        scratch, total, err_flag, cap);
    } else {
      scratch = nullptr;
      k_neighbors<0><<<nblk(N * 32, 256), 256, 0, st>>>(N, g, pos_s, wrap_s, cellid_s, cell_start, deg, nullptr,
                                                        nullptr, total, err_flag, 0);
    }
    ctx->launches += 4;
  }
  unsigned long long total_h = 0;
  int err_h = 0, sp_h[2] = {0, 0};
  if (cudaMemcpyAsync(&total_h, total, sizeof(total_h), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaMemcpyAsync(sp_h, sp_range, sizeof(sp_h), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaMemcpyAsync(&err_h, err_flag, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess) {
    ctx->set_error(std::string("graph build (count): ") + cudaGetErrorString(cudaGetLastError()));
    return fail(MLIP_ERR_CUDA);
  }
  if (err_h & 1) { ctx->set_error("image shift outside [-127,127]"); return fail(MLIP_ERR_OVERFLOW); }
  if (total_h >= (1ull << 31)) { ctx->set_error("number of edges >= 2^31"); return fail(MLIP_ERR_OVERFLOW); }
  const int64_t E = (int64_t)total_h;
  G->E = E;
  G->species_max = sp_h[0]; G->species_min = -sp_h[1];
  G_TRY(mlip_exclusive_scan_i32(ctx, deg, G->rowptr, N, nullptr));
  G_TRY(ctx->alloc(&keys, E)); G_TRY(ctx->alloc(&G->recv, E)); G_TRY(ctx->alloc(&G->send, E));
  G_TRY(ctx->alloc(&G->shift, E)); G_TRY(ctx->alloc(&G->rev, E)); G_TRY(ctx->alloc(&G->rvec, E));
  if (E > 0) {
    if (scratch && !(err_h & 4))
      k_compact_keys<<<nblk(N * 32, 256), 256, 0, st>>>(N, cap, G->rowptr, scratch, keys);
    else
      k_neighbors<1><<<nblk(N * 32, 256), 256, 0, st>>>(N, g, pos_s, wrap_s, cellid_s, cell_start, nullptr,
                                                        G->rowptr, keys, nullptr, err_flag, 0);
    k_sort_rows<<<nblk(N, 4), 128, 0, st>>>(N, G->rowptr, keys);
    k_finalize_edges<<<nblk(N * 32, 256), 256, 0, st>>>(N, g, pos_s, G->rowptr, keys, G->recv, G->send, G->shift,
                                                        G->rvec);
    k_reverse<<<nblk(E, 256), 256, 0, st>>>(E, G->rowptr, G->recv, keys, G->rev, ctx->dev_status);
    ctx->launches += 4;
  }
  ctx->free(frac); ctx->free(wrap); ctx->free(cellid); ctx->free(cell_count); ctx->free(cell_start);
  ctx->free(order); ctx->free(pos_s); ctx->free(wrap_s); ctx->free(cellid_s); ctx->free(deg);
  ctx->free(total); ctx->free(keys); ctx->free(scratch); ctx->free(sp_range);
  cudaError_t e = cudaGetLastError();
  ctx->free(err_flag);
  if (e != cudaSuccess) { ctx->set_error(std::string("graph build: ") + cudaGetErrorString(e)); return fail(MLIP_ERR_CUDA); }
#undef G_TRY
  *out = G;
  return MLIP_OK;
}

extern "C" int mlip_graph_num_edges(const mlip_graph* g, int64_t* n_edges) {
  if (!g || !n_edges) return MLIP_ERR_INVALID_ARG;
  *n_edges = g->E;
  return MLIP_OK;
}

extern "C" void mlip_graph_destroy(mlip_graph* G) {
  if (!G) return;
  mlip_ctx* c = G->ctx;
  c->free(G->perm); c->free(G->frac); c->free(G->species); c->free(G->rowptr); c->free(G->recv);
  c->free(G->send); c->free(G->shift); c->free(G->rev); c->free(G->rvec);
  delete G;
}

extern "C" int mlip_graph_export_edges(mlip_ctx* ctx, const mlip_graph* G, int32_t* recv_dev, int32_t* send_dev,
                                       int32_t* shift_dev) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!G || (G->E > 0 && (!recv_dev || !send_dev || !shift_dev))) {
    ctx->set_error("mlip_graph_export_edges: invalid argument");
    return MLIP_ERR_INVALID_ARG;
  }
  const int64_t N = G->N, E = G->E;
  if (E == 0) return MLIP_OK;
  cudaStream_t st = ctx->stream;
  int32_t *inv = nullptr, *deg_o = nullptr, *rowptr_o = nullptr;
  unsigned long long* keys = nullptr;
  MLIP_TRY(ctx->alloc(&inv, N)); MLIP_TRY(ctx->alloc(&deg_o, N)); MLIP_TRY(ctx->alloc(&rowptr_o, N + 1));
  MLIP_TRY(ctx->alloc(&keys, E));
  k_invert_perm<<<nblk(N, 256), 256, 0, st>>>(G->perm, N, inv);
  k_export_deg<<<nblk(N, 256), 256, 0, st>>>(inv, G->rowptr, N, deg_o);
  ctx->launches += 2;
  MLIP_TRY(mlip_exclusive_scan_i32(ctx, deg_o, rowptr_o, N, nullptr));
  k_export_keys<<<nblk(N * 32, 256), 256, 0, st>>>(N, inv, G->perm, G->rowptr, G->send, G->shift, rowptr_o, keys);
  k_sort_rows<<<nblk(N, 4), 128, 0, st>>>(N, rowptr_o, keys);
  k_export_decode<<<nblk(N * 32, 256), 256, 0, st>>>(N, rowptr_o, keys, recv_dev, send_dev, shift_dev);
  ctx->launches += 3;
  ctx->free(inv); ctx->free(deg_o); ctx->free(rowptr_o); ctx->free(keys);
  MLIP_CUDA_CHECK(ctx, cudaGetLastError());
  return MLIP_OK;
}
