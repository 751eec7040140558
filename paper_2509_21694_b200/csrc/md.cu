// On-device molecular dynamics driver (the use the paper builds the partitioned evaluation for: ns-scale MD of
// 10^5..10^6 atoms): velocity-Verlet NVE and Langevin (BAOAB, reading R20; the paper runs ASE's
// Langevin integrator) integration with the whole step -- neighbour list, partition, energy and
// forces, kicks, drift, thermostat, kinetic energy -- on the GPU; the host only sequences launches.
// Positions and velocities stay in float64 (the graph builder's predicate is float64, reading R10); forces are the
// float32 output of mlip_energy_forces. Units: Angstrom, fs, amu, eV (1 eV/A/amu = 9.648533e-3 A/fs^2).
#include <string.h>
#include "common.cuh"
#include "skin.cuh"

namespace {
constexpr double ACC_UNIT = 9.648533e-3;  // (eV/A)/amu -> A/fs^2

inline unsigned nblk(int64_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// v += (dt/2) a ; optionally x += dt v   (a = ACC_UNIT F / m)
__global__ void k_vv_kick(int64_t N, double half_dt, double drift_dt, const float* __restrict__ F,
                          const double* __restrict__ mass, double* __restrict__ vel, double* __restrict__ pos) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 3 * N) return;
  const double v = vel[i] + half_dt * ACC_UNIT * (double)F[i] / mass[i / 3];
  vel[i] = v;
  if (drift_dt != 0.0) pos[i] += drift_dt * v;
}

// ---- Langevin thermostat: Philox4x32-10 normals, a pure function of (seed, step, atom) --------------------------------
constexpr double KB_EV = 8.617333262e-5;  // eV/K
__device__ __forceinline__ void philox4x32_10(uint32_t (&c)[4], uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c[0]), lo0 = 0xD2511F53u * c[0];
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c[2]), lo1 = 0xCD9E8D57u * c[2];
    const uint32_t n0 = hi1 ^ c[1] ^ k0, n2 = hi0 ^ c[3] ^ k1;
    c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
}
// B A O A of one BAOAB step for atom i (the closing B is k_vv_kick after the force evaluation):
//   v += (dt/2) a ; x += (dt/2) v ; v = c1 v + c2 sqrt(kB T / m) xi ; x += (dt/2) v
__global__ void __launch_bounds__(256) k_baoab_pre(int64_t N, double dt, double c1, double c2, double kT, uint64_t seed,
                                                   uint32_t step, const float* __restrict__ F, const double* __restrict__ mass,
                                                   double* __restrict__ vel, double* __restrict__ pos) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  uint32_t c[4] = {(uint32_t)i, step, 0u, 0u};
  philox4x32_10(c, (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32));
  const double u1 = ((double)c[0] + 0.5) * 2.3283064365386963e-10, u2 = ((double)c[1] + 0.5) * 2.3283064365386963e-10;
  const double u3 = ((double)c[2] + 0.5) * 2.3283064365386963e-10, u4 = ((double)c[3] + 0.5) * 2.3283064365386963e-10;
  const double ra = sqrt(-2.0 * log(u1)), rb = sqrt(-2.0 * log(u3));
  double s2, c2pi, s4, c4pi;
  sincospi(2.0 * u2, &s2, &c2pi);
  sincospi(2.0 * u4, &s4, &c4pi);
  const double xi[3] = {ra * c2pi, ra * s2, rb * c4pi};
  const double m = mass[i], sig = sqrt(kT * ACC_UNIT / m);
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    double v = vel[3 * i + k] + 0.5 * dt * ACC_UNIT * (double)F[3 * i + k] / m;
    double x = pos[3 * i + k] + 0.5 * dt * v;
    v = c1 * v + c2 * sig * xi[k];
    x += 0.5 * dt * v;
    vel[3 * i + k] = v;
    pos[3 * i + k] = x;
  }
}

// kinetic energy (eV) = 1/2 sum m v^2 / ACC_UNIT: float64 per-block partials, then one block (deterministic)
__global__ void __launch_bounds__(256) k_kinetic_partial(int64_t N, const double* __restrict__ mass,
                                                         const double* __restrict__ vel, double* __restrict__ partial) {
  __shared__ double sh[256];
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
    const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
    s += mass[i] * ((vx * vx + vy * vy) + vz * vz);
  }
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int k = 128; k > 0; k >>= 1) {
    if (threadIdx.x < k) sh[threadIdx.x] += sh[threadIdx.x + k];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
// total[step] = E_pot + kinetic
__global__ void k_total_energy(int n_partial, const double* __restrict__ partial, const double* __restrict__ e_pot,
                               double* __restrict__ out) {
  if (threadIdx.x != 0) return;
  double s = 0.0;
  for (int i = 0; i < n_partial; ++i) s += partial[i];
  out[0] = e_pot[0] + 0.5 * s / ACC_UNIT;
}

// Graph -> partition -> E, F at the current positions. skin = 0: everything is rebuilt on every call. skin > 0: the candidate
// graph (r_c + skin) and its partition are kept until an atom has moved more than skin/2 (skin.cu); the per-step work --
// filter, layers, reverse pass, force assembly -- has fixed launch dimensions between rebuilds and can be replayed from a
// CUDA graph.
__global__ void k_md_check_finite(int64_t n, const float* __restrict__ F, const double* __restrict__ energy, int* __restrict__ status) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = i < n && !isfinite(F[i]);
  if (i == 0) bad = bad || !isfinite(energy[0]);
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(status, MLIP_DEV_NONFINITE);
}

struct MdEvaluator {
  mlip_ctx* ctx; const mlip_model* M; int L; const double* pos; const double* cell; const int32_t* species; int64_t N;
  int grid[3]; double halo; int precision; double skin; bool use_graph; double* e_pot; float* F;
  int64_t n_rebuilds = 0, n_replays = 0;
  // skin mode
  mlip_graph* Gc = nullptr;
  mlip_part* Pc = nullptr;
  std::vector<SkinSub> subs;
  double* pos0 = nullptr;
  int* flag = nullptr;
  cudaGraphExec_t exec = nullptr;
  bool capture_failed = false;
  std::string capture_error;
  MdEvaluator(mlip_ctx* c, const mlip_model* m, int L_, const double* p, const double* cell_, const int32_t* sp, int64_t n,
              const int g[3], double h, int prec, double skin_, bool graph, double* e, float* f)
      : ctx(c), M(m), L(L_), pos(p), cell(cell_), species(sp), N(n), halo(h), precision(prec), skin(skin_), use_graph(graph),
        e_pot(e), F(f) {
    grid[0] = g[0]; grid[1] = g[1]; grid[2] = g[2];
  }
  ~MdEvaluator() { drop(); ctx->free(pos0); ctx->free(flag); }
  bool split() const { return grid[0] > 1 || grid[1] > 1 || grid[2] > 1; }
  void drop() {
    if (exec) { cudaGraphExecDestroy(exec); exec = nullptr; }
    for (auto& k : subs) k.release(ctx);
    subs.clear();
    mlip_part_destroy(Pc); Pc = nullptr;
    mlip_graph_destroy(Gc); Gc = nullptr;
  }
  int evaluate() { return skin > 0.0 ? evaluate_skin() : evaluate_rebuild(); }

  int evaluate_rebuild() {
    mlip_graph* G = nullptr;
    mlip_part* P = nullptr;
    int s = mlip_build_graph(ctx, pos, cell, species, N, (double)M->h.r_cut, &G);
    if (s == MLIP_OK && split()) s = mlip_partition_grid(ctx, G, grid, halo, &P);
    if (s == MLIP_OK) s = mlip_energy_forces(ctx, M, L, G, P, precision, e_pot, F, nullptr);
    mlip_part_destroy(P);
    mlip_graph_destroy(G);
    ++n_rebuilds;
    return s;
  }

  int rebuild() {
    drop();
    const double r_c = (double)M->h.r_cut;
    MLIP_TRY(mlip_build_graph(ctx, pos, cell, species, N, r_c + skin, &Gc));
    if (N > 0 && (Gc->species_min < 0 || Gc->species_max >= M->h.n_species)) {
      ctx->set_error("species outside [0, n_species) of the model");
      return MLIP_ERR_INVALID_ARG;
    }
    if (split()) {
      if (halo < (double)L * r_c * (1.0 - 1e-12)) {
        ctx->set_error("halo < L * r_cut: sub-graphs would not keep the K-hop neighbourhood of their root atoms");
        return MLIP_ERR_HALO_TOO_SMALL;
      }
      MLIP_TRY(mlip_partition_grid_ex(ctx, Gc, grid, halo + skin, halo, r_c, true, true, &Pc));
      subs.resize(Pc->subs.size());
      for (size_t k = 0; k < subs.size(); ++k) MLIP_TRY(mlip_skin_sub_create(ctx, Gc, &Pc->subs[k], &subs[k]));
    } else {
      subs.resize(1);
      MLIP_TRY(mlip_skin_sub_create(ctx, Gc, nullptr, &subs[0]));
    }
    if (!pos0) MLIP_TRY(ctx->alloc(&pos0, 3 * N));
    cudaMemcpyAsync(pos0, pos, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, ctx->stream);
    ++n_rebuilds;
    return MLIP_OK;
  }

  // filter + evaluate every sub-domain at the current positions (fixed launch dimensions)
  int step_eager() {
    cudaStream_t st = ctx->stream;
    cudaMemsetAsync(F, 0, sizeof(float) * 3 * N, st);
    cudaMemsetAsync(e_pot, 0, sizeof(double), st);
    for (auto& k : subs) {
      MLIP_TRY(mlip_skin_filter(ctx, k, pos, cell, (double)M->h.r_cut));
      MLIP_TRY(mlip_eval_subgraph(ctx, M, L, k.g, precision, e_pot, F, nullptr, nullptr));
    }
    if (N > 0) {
      k_md_check_finite<<<nblk(3 * N, 256), 256, 0, st>>>(3 * N, F, e_pot, ctx->dev_status);
      ctx->launches++;
    }
    return MLIP_OK;
  }

  int evaluate_skin() {
    cudaStream_t st = ctx->stream;
    bool need = Gc == nullptr;
    if (!need) {
      if (!flag) MLIP_TRY(ctx->alloc(&flag, 1));
      MLIP_TRY(mlip_skin_moved(ctx, N, pos, pos0, skin, flag));
      int h = 0;
      MLIP_CUDA_CHECK(ctx, cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, st));
      MLIP_CUDA_CHECK(ctx, cudaStreamSynchronize(st));
      need = h != 0;
    }
    if (need) MLIP_TRY(rebuild());
    if (use_graph && !capture_failed) {
      if (!exec) {
        // capture one step: kernels, memsets and stream-ordered allocations become graph nodes
        const bool was_profiling = ctx->profiling;
        ctx->profiling = false;
        cudaGraph_t graph = nullptr;
        int s = MLIP_OK;
        // the legacy default stream cannot be captured: record on a private stream, replay on the context stream
        cudaStream_t cap = nullptr;
        if (cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) == cudaSuccess) {
          ctx->stream = cap;
          cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
          if (e == cudaSuccess) {
            s = step_eager();
            e = cudaStreamEndCapture(cap, &graph);
          }
          ctx->stream = st;
          if (s == MLIP_OK && e == cudaSuccess && graph) e = cudaGraphInstantiate(&exec, graph, 0);
          if (s != MLIP_OK || e != cudaSuccess) {
            exec = nullptr;
            capture_error = e != cudaSuccess ? cudaGetErrorString(e) : ctx->err;
          }
          if (graph) cudaGraphDestroy(graph);
          cudaStreamDestroy(cap);
        }
        ctx->profiling = was_profiling;
        cudaGetLastError();
        if (!exec) capture_failed = true;   // fall back to plain launches for the rest of the run
      }
      if (exec) {
        MLIP_CUDA_CHECK(ctx, cudaGraphLaunch(exec, st));
        ++n_replays;
        return MLIP_OK;
      }
    }
    return step_eager();
  }
};
}  // namespace

extern "C" int mlip_md_run(mlip_ctx* ctx, const mlip_model* M, int L, double* pos_dev, double* vel_dev,
                           const double* mass_dev, const double* cell_host, const int32_t* species_dev, int64_t N,
                           const int grid[3], double halo, int precision, const mlip_md_params* prm,
                           double* total_energy_host, mlip_md_stats* stats) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!M || (N > 0 && (!pos_dev || !vel_dev || !mass_dev || !species_dev)) || !cell_host || !grid || !prm || N < 0 || prm->n_steps < 0 ||
      !(prm->dt > 0.0) || (prm->thermostat != MLIP_MD_NVE && prm->thermostat != MLIP_MD_LANGEVIN) || !(prm->skin >= 0.0)) {
    ctx->set_error("mlip_md_run: invalid argument");
    return MLIP_ERR_INVALID_ARG;
  }
  const bool langevin = prm->thermostat == MLIP_MD_LANGEVIN;
  if (langevin && (!(prm->temperature >= 0.0) || !(prm->friction >= 0.0))) {
    ctx->set_error("mlip_md_run: Langevin needs temperature >= 0 and friction >= 0");
    return MLIP_ERR_INVALID_ARG;
  }
  if (prm->cuda_graph && !(prm->skin > 0.0)) {
    ctx->set_error("mlip_md_run: cuda_graph = 1 needs skin > 0 (launch dimensions are only fixed between rebuilds)");
    return MLIP_ERR_INVALID_ARG;
  }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  const int n_steps = prm->n_steps;
  const double dt = prm->dt;
  const int nb = (int)(N < 148 * 4 * 256 ? (N + 255) / 256 : 148 * 4);
  float* F = nullptr;
  double *e_pot = nullptr, *partial = nullptr, *e_tot = nullptr;
  Scratch tmp(ctx);
  MLIP_TRY(tmp.get(&F, 3 * N)); MLIP_TRY(tmp.get(&e_pot, 1)); MLIP_TRY(tmp.get(&partial, nb > 0 ? nb : 1));
  MLIP_TRY(tmp.get(&e_tot, n_steps + 1));
  MdEvaluator ev(ctx, M, L, pos_dev, cell_host, species_dev, N, grid, halo, precision, prm->skin, prm->cuda_graph != 0, e_pot, F);
  const double c1 = langevin ? exp(-prm->friction * dt) : 1.0;
  const double c2 = langevin ? sqrt(1.0 - c1 * c1) : 0.0;
  auto record = [&](int step) {
    if (N > 0) k_kinetic_partial<<<nb, 256, 0, st>>>(N, mass_dev, vel_dev, partial);
    k_total_energy<<<1, 32, 0, st>>>(N > 0 ? nb : 0, partial, e_pot, e_tot + step);
    ctx->launches += 2;
  };
  int status = ev.evaluate();
  cudaEvent_t t0 = ctx->get_event(), t1 = ctx->get_event();
  cudaEventRecord(t0, st);
  for (int step = 0; step < n_steps && status == MLIP_OK; ++step) {
    record(step);
    if (N > 0) {
      if (langevin && c2 > 0.0)
        k_baoab_pre<<<nblk(N, 256), 256, 0, st>>>(N, dt, c1, c2, KB_EV * prm->temperature, prm->seed, (uint32_t)step, F, mass_dev,
                                                 vel_dev, pos_dev);
      else
        k_vv_kick<<<nblk(3 * N, 256), 256, 0, st>>>(N, 0.5 * dt, dt, F, mass_dev, vel_dev, pos_dev);
      ctx->launches++;
    }
    status = ev.evaluate();
    if (status == MLIP_OK && N > 0) {
      k_vv_kick<<<nblk(3 * N, 256), 256, 0, st>>>(N, 0.5 * dt, 0.0, F, mass_dev, vel_dev, pos_dev);
      ctx->launches++;
    }
  }
  cudaEventRecord(t1, st);
  if (status == MLIP_OK) {
    record(n_steps);
    if (total_energy_host)
      cudaMemcpyAsync(total_energy_host, e_tot, sizeof(double) * (n_steps + 1), cudaMemcpyDeviceToHost, st);
  }
  cudaError_t e = cudaStreamSynchronize(st);
  float ms = 0.f;
  if (e == cudaSuccess) cudaEventElapsedTime(&ms, t0, t1);
  ctx->event_pool.push_back(t0); ctx->event_pool.push_back(t1);
  if (stats) { stats->n_rebuilds = ev.n_rebuilds; stats->n_graph_replays = ev.n_replays; stats->ms_total = ms; }
  if (ev.capture_failed) ctx->set_error("md: CUDA-graph capture failed (" + ev.capture_error + "); the run used plain launches");
  if (status != MLIP_OK) return status;
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) { ctx->set_error(std::string("md: ") + cudaGetErrorString(e)); return MLIP_ERR_CUDA; }
  return mlip_take_dev_status(ctx);
}

extern "C" int mlip_md_nve(mlip_ctx* ctx, const mlip_model* M, int L, double* pos_dev, double* vel_dev,
                           const double* mass_dev, const double* cell_host, const int32_t* species_dev, int64_t N,
                           const int grid[3], double halo, int precision, double dt, int n_steps,
                           double* total_energy_host) {
  mlip_md_params p;
  memset(&p, 0, sizeof(p));
  p.dt = dt; p.n_steps = n_steps; p.thermostat = MLIP_MD_NVE;
  return mlip_md_run(ctx, M, L, pos_dev, vel_dev, mass_dev, cell_host, species_dev, N, grid, halo, precision, &p,
                     total_energy_host, nullptr);
}
