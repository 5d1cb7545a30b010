// Host-side plumbing shared by the translation units of wt_solve_H (not part of the ABI):
//   solve.cu             argument checks, static tables -> workspace, descriptors, dispatch
//   solve_chain.cu       one kernel per phase and substep, captured in a CUDA graph (any 2^a 3^b grid, any pad count,
//                        lock-step batches)
//   solve_persistent.cu  one cooperative launch per output step (power-of-two grids of the BASELINE configs)
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "geometry.h"
#include "solve_common.cuh"

namespace wt {

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }
bool env_flag(const char* name);

// pads of one geometry grouped by (layer, x); perm[i] = index (in the handle's pad order) of the
// i-th pad in group order; the device holds every per-pad array in group order
struct PadGroups {
  std::vector<int> grp_x, grp_layer, grp_off, perm, layer_goff, pad_y, pad_x, pad_l, layer_poff;
  std::vector<double> pad_pot, ainv;
  int max_per_layer = 0;
};
PadGroups make_groups(const wt_geometry* g);


// Offsets of one geometry's region inside the workspace: static tables [0, static_bytes), then state.
struct Layout {
  size_t sig_id, sig_t, sdt, gt, gzt, ainv, pad_pot, pad_y, pad_x, pad_l, grp_x, grp_layer, grp_off, layer_goff;
  size_t kxd, kyd, kzd, kxf, kyf, kzf, twx, twy, twz, twxd, twyd, twzd;
  size_t static_bytes;
  size_t rhat, rhat_prev, v0, v1, m0, m1, m2, e0, e1, pl, pl_e, rhs, q, qh, part, ctl, stage;
#ifdef WTIDE_DEBUG
  size_t dbg;          // 256 KB of clock stamps (timing experiments)
#endif
  size_t total;
};
Layout make_layout(const wt_geometry* g);

// One geometry as the solvers see it
struct GeomHost {
  const wt_geometry* g;
  const PadGroups* pg;
  Layout lo;
  char* base;          // device address of the geometry's region
  GeomDev dev;
};

struct SolveStats { long long launches = 0; };

// solve_chain.cu: lock-step batch through the per-substep kernel chain.  dstep = device int (zeroed here).
int chain_solve(std::vector<GeomHost>& geoms, GridDev gd, int* dstep, cudaStream_t st, SolveStats* stats);
void chain_describe(const wt_geometry* g, std::string* out);

// solve_persistent.cu
bool persistent_eligible(const wt_geometry* g, int n_pads);
int persistent_solve(GeomHost& gh, GridDev gd, cudaStream_t st, SolveStats* stats);
void persistent_describe(const wt_geometry* g, std::string* out);

}  // namespace wt
