// Canonical float64 edge vector and squared length of O1 / reading R10: fixed operation order, no FMA
// contraction -- t = (nx a1 + ny a2) + nz a3 ; r = (x_j - x_i) + t ; d2 = (rx rx + ry ry) + rz rz. Shared by the graph
// builder (graph.cu) and the Verlet-skin filter (skin.cu) so that both accept exactly the same edges.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

__device__ __forceinline__ double canonical_rvec(const double* __restrict__ cell /*[9] rows a1,a2,a3*/, int nx, int ny, int nz,
                                                 double xi, double yi, double zi, double xj, double yj, double zj,
                                                 double& rx, double& ry, double& rz) {
  const double fx = (double)nx, fy = (double)ny, fz = (double)nz;
  const double tx = __dadd_rn(__dadd_rn(__dmul_rn(fx, cell[0]), __dmul_rn(fy, cell[3])), __dmul_rn(fz, cell[6]));
  const double ty = __dadd_rn(__dadd_rn(__dmul_rn(fx, cell[1]), __dmul_rn(fy, cell[4])), __dmul_rn(fz, cell[7]));
  const double tz = __dadd_rn(__dadd_rn(__dmul_rn(fx, cell[2]), __dmul_rn(fy, cell[5])), __dmul_rn(fz, cell[8]));
  rx = __dadd_rn(__dadd_rn(xj, -xi), tx);
  ry = __dadd_rn(__dadd_rn(yj, -yi), ty);
  rz = __dadd_rn(__dadd_rn(zj, -zi), tz);
  return __dadd_rn(__dadd_rn(__dmul_rn(rx, rx), __dmul_rn(ry, ry)), __dmul_rn(rz, rz));
}
