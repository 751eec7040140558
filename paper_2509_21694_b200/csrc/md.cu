// On-device molecular dynamics driver (the use the paper builds the partitioned evaluation for: ns-scale MD of
// 10^5..10^6 atoms): velocity-Verlet NVE integration with the whole step -- neighbour list,
// partition, energy and forces, kicks and drift, kinetic energy -- on the GPU; the host only sequences launches.
// Positions and velocities stay in float64 (the graph builder's predicate is float64, reading R10); forces are the
// float32 output of mlip_energy_forces. Units: Angstrom, fs, amu, eV (1 eV/A/amu = 9.648533e-3 A/fs^2).
#include "common.cuh"

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
}  // namespace

extern "C" int mlip_md_nve(mlip_ctx* ctx, const mlip_model* M, int L, double* pos_dev, double* vel_dev,
                           const double* mass_dev, const double* cell_host, const int32_t* species_dev, int64_t N,
                           const int grid[3], double halo, int precision, double dt, int n_steps,
                           double* total_energy_host) {
  if (!ctx) return MLIP_ERR_INVALID_ARG;
  if (!M || !pos_dev || !vel_dev || !mass_dev || !cell_host || !species_dev || !grid || N < 0 || n_steps < 0 || !(dt > 0.0)) {
    ctx->set_error("mlip_md_nve: invalid argument");
    return MLIP_ERR_INVALID_ARG;
  }
  MLIP_CUDA_CHECK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  const bool split = grid[0] > 1 || grid[1] > 1 || grid[2] > 1;
  const int nb = (int)(N < 148 * 4 * 256 ? (N + 255) / 256 : 148 * 4);
  float* F = nullptr;
  double *e_pot = nullptr, *partial = nullptr, *e_tot = nullptr;
  Scratch tmp(ctx);
  MLIP_TRY(tmp.get(&F, 3 * N)); MLIP_TRY(tmp.get(&e_pot, 1)); MLIP_TRY(tmp.get(&partial, nb > 0 ? nb : 1));
  MLIP_TRY(tmp.get(&e_tot, n_steps + 1));
  int status = MLIP_OK;
  auto evaluate = [&]() {  // graph -> partition -> E, F at the current positions
    mlip_graph* G = nullptr;
    mlip_part* P = nullptr;
    int s = mlip_build_graph(ctx, pos_dev, cell_host, species_dev, N, (double)M->h.r_cut, &G);
    if (s == MLIP_OK && split) s = mlip_partition_grid(ctx, G, grid, halo, &P);
    if (s == MLIP_OK) s = mlip_energy_forces(ctx, M, L, G, P, precision, e_pot, F, nullptr);
    mlip_part_destroy(P);
    mlip_graph_destroy(G);
    return s;
  };
  auto record = [&](int step) {
    if (N > 0) k_kinetic_partial<<<nb, 256, 0, st>>>(N, mass_dev, vel_dev, partial);
    k_total_energy<<<1, 32, 0, st>>>(N > 0 ? nb : 0, partial, e_pot, e_tot + step);
    ctx->launches += 2;
  };
  status = evaluate();
  for (int step = 0; step < n_steps && status == MLIP_OK; ++step) {
    record(step);
    if (N > 0) {
      k_vv_kick<<<nblk(3 * N, 256), 256, 0, st>>>(N, 0.5 * dt, dt, F, mass_dev, vel_dev, pos_dev);
      ctx->launches++;
    }
    status = evaluate();
    if (status == MLIP_OK && N > 0) {
      k_vv_kick<<<nblk(3 * N, 256), 256, 0, st>>>(N, 0.5 * dt, 0.0, F, mass_dev, vel_dev, pos_dev);
      ctx->launches++;
    }
  }
  if (status == MLIP_OK) {
    record(n_steps);
    if (total_energy_host)
      cudaMemcpyAsync(total_energy_host, e_tot, sizeof(double) * (n_steps + 1), cudaMemcpyDeviceToHost, st);
  }
  cudaError_t e = cudaStreamSynchronize(st);
  if (status != MLIP_OK) return status;
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) { ctx->set_error(std::string("md: ") + cudaGetErrorString(e)); return MLIP_ERR_CUDA; }
  return mlip_take_dev_status(ctx);
}
