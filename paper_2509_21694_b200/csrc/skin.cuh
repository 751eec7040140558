// Verlet-skin mode of the MD driver: one sub-domain (or the whole box) as a fixed candidate list plus the exact,
// re-filtered edge arrays of the current step (see skin.cu).
#pragma once
#include "common.cuh"

struct SkinSub {
  int64_t n = 0, E_cap = 0;
  // candidate list, borrowed from the candidate graph / partition (alive as long as they are)
  const int32_t *c_rowptr = nullptr, *c_send = nullptr, *c_rev = nullptr;
  int32_t *aid = nullptr;      // [n] caller atom index of every local atom
  int32_t *c_shift = nullptr;  // [E_cap] packed image shifts of the candidates
  // exact graph of the current step (capacity E_cap)
  int32_t *rowptr = nullptr, *recv = nullptr, *send = nullptr, *rev = nullptr, *newpos = nullptr, *cand = nullptr, *deg = nullptr;
  float4* rvec = nullptr;
  SubGraph g;                  // what mlip_eval_subgraph gets (dyn = true, gid = aid)
  void release(mlip_ctx* ctx);
};

// S == nullptr: the whole (unpartitioned) candidate graph G
int mlip_skin_sub_create(mlip_ctx* ctx, const mlip_graph* G, const PartSub* S, SkinSub* out);
int mlip_skin_filter(mlip_ctx* ctx, const SkinSub& k, const double* pos_dev, const double* cell_host, double r_cut);
int mlip_skin_moved(mlip_ctx* ctx, int64_t N, const double* pos_dev, const double* pos0_dev, double skin, int* flag_dev);
