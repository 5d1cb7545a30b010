// wt_solve_H through the per-substep kernel chain: one kernel per phase (boundary adjust, xy-planes, z-lines) and
// Euler substep, the kernels of one output step captured once into a CUDA graph and replayed nt-1 times.
// This is the path for every 2^a 3^b grid, for pad sets of any size and for lock-step batches; the power-of-two
// grids of the BASELINE configs run on the persistent kernel of solve_persistent.cu instead (WTIDE_CHAIN=1 forces
// the chain).  Method and phase split: see solve.cu.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

#include "solve_boundary.cuh"
#include "solve_fast.cuh"
#include "solve_generic.cuh"
#include "solve_plan.h"

namespace wt {
namespace {

int pick_ty(int y2) {
  const int cand[6] = {8, 6, 4, 3, 2, 1};
  for (int c : cand)
    if (y2 % c == 0) return c;
  return 1;
}

#define CK(call)                                                                              \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      wt_set_error(std::string("wt_solve_H (chain): ") + cudaGetErrorString(e_) + " at " #call);      \
      return WT_ECUDA;                                                                        \
    }                                                                                         \
  } while (0)

// One launch: optional thread-block cluster along x, optional programmatic dependent launch (PDL).
template <typename... KArgs, typename... Args>
cudaError_t launch(void (*fn)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, int cluster,
                   Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[2];
  int n = 0;
  if (cluster > 1) {
    at[n].id = cudaLaunchAttributeClusterDimension;
    at[n].val.clusterDim.x = cluster; at[n].val.clusterDim.y = 1; at[n].val.clusterDim.z = 1;
    ++n;
  }
  if (pdl) {
    at[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[n].val.programmaticStreamSerializationAllowed = 1;
    ++n;
  }
  cfg.attrs = at; cfg.numAttrs = n;
  return cudaLaunchKernelEx(&cfg, fn, std::forward<Args>(args)...);
}

// ---- kernel selection ---------------------------------------------------------------------------
using PlaneFn = void (*)(const GeomBatch, GridDev, int);
using LineFn = void (*)(const GeomBatch, GridDev, int, int);

struct Plan {
  PlaneFn plane_step = nullptr, plane_emit = nullptr;
  dim3 plane_block;
  size_t plane_smem = 0;
  bool plane_fast = false;     // one CTA per (z, component); staging layout [z][y][x] instead of [z][x][y]
  LineFn line_step = nullptr, line_init = nullptr, line_delta = nullptr;   // <J>, <>, <DELTA>
  dim3 line_grid, line_block;
  size_t line_smem = 0;
  bool line_fast = false;
  int ty = 1;
};

template <int N, int E>
void set_plane(Plan& p) {
  p.plane_step = k_plane_fast<N, E, false>;
  p.plane_emit = k_plane_fast<N, E, true>;
  p.plane_block = dim3(N * N / (2 * E));
  p.plane_smem = (size_t)2 * PlaneCfg<N>::BUF * sizeof(float2);
  p.plane_fast = true;
}

template <int NZ, int E, int TYL, int LT>
void set_line_lt(Plan& p, int nx, int y2) {
  using C = PencilCfg<NZ, E, TYL>;
  p.line_step = k_pencil<NZ, E, TYL, LT, true, false>;
  p.line_init = k_pencil<NZ, E, TYL, LT, false, false>;
  p.line_delta = k_pencil<NZ, E, TYL, LT, false, true>;
  p.line_grid = dim3(nx * (y2 / TYL));
  p.line_block = dim3(C::THREADS);
  p.line_smem = (size_t)2 * C::FIELD * sizeof(float2) + (size_t)LT * TYL * C::T * sizeof(double2);
  p.line_fast = true;
  p.ty = TYL;
}
template <int NZ, int E, int TYL, int LT>
void set_line2_lt(Plan& p, int nx, int y2) {
  using C = PencilCfg<NZ, E, TYL>;
  p.line_step = k_pencil2<NZ, E, TYL, LT, true, false>;
  p.line_init = k_pencil2<NZ, E, TYL, LT, false, false>;
  p.line_delta = k_pencil2<NZ, E, TYL, LT, false, true>;
  p.line_grid = dim3(nx * (y2 / TYL));
  p.line_block = dim3(2 * C::THREADS);
  p.line_smem = (size_t)2 * C::FIELD * sizeof(float2) + (size_t)2 * NZ * TYL * sizeof(float2) +
                (size_t)LT * TYL * 2 * C::T * sizeof(double2);
  p.line_fast = true;
  p.ty = TYL;
}
template <int NZ, int E, int TYL>
void set_line(Plan& p, int nx, int y2, int L) {
  if (!env_flag("WTIDE_PENCIL1")) {
    if (L <= 2) set_line2_lt<NZ, E, TYL, 2>(p, nx, y2);
    else set_line2_lt<NZ, E, TYL, kMaxLayers>(p, nx, y2);
    return;
  }
  if (L <= 2) set_line_lt<NZ, E, TYL, 2>(p, nx, y2);
  else set_line_lt<NZ, E, TYL, kMaxLayers>(p, nx, y2);
}

Plan make_plan(int nx, int ny, int nz, int L, bool force_generic) {
  Plan p;
  const int y2 = ny / 2;
  if (!force_generic && nx == ny) {
    if (nx == 32) set_plane<32, 8>(p);
    else if (nx == 64) set_plane<64, 8>(p);
    else if (nx == 128) set_plane<128, 16>(p);
    else if (nx == 96) set_plane<96, 24>(p);       // configs[4]: radix-3 register transform (dft24 x dft4)
  }
  if (!p.plane_fast) {
    p.plane_step = k_plane<false>;
    p.plane_emit = k_plane<true>;
    p.plane_block = dim3(256);
    p.plane_smem = (size_t)2 * (nx / 2) * (ny + 1) * sizeof(float2) + (size_t)(nx + ny) * sizeof(float2);
  }
  if (!force_generic) {
    if (nz == 256 && y2 % 8 == 0) set_line<256, 16, 8>(p, nx, y2, L);
    else if (nz == 128 && y2 % 16 == 0) set_line<128, 16, 16>(p, nx, y2, L);
    else if (nz == 64 && y2 % 16 == 0) set_line<64, 8, 16>(p, nx, y2, L);
    else if (nz == 32 && y2 % 16 == 0) set_line<32, 8, 16>(p, nx, y2, L);
  }
  if (!p.line_fast) {
    p.ty = pick_ty(y2);
    p.line_step = k_spectral<true, false>;
    p.line_init = k_spectral<false, false>;
    p.line_delta = k_spectral<false, true>;
    p.line_grid = dim3(nx * (y2 / p.ty));
    p.line_block = dim3(32 * p.ty);
    p.line_smem = (size_t)3 * nz * p.ty * sizeof(float2) + (size_t)std::max(1, L) * p.ty * 32 * sizeof(double2) + (size_t)nz * (sizeof(float2) + sizeof(double2) + sizeof(double));
  }
  return p;
}

}  // namespace

void chain_describe(const wt_geometry* g, std::string* out) {
  const Plan p = make_plan(g->nx, g->ny, g->nz, (int)g->layers.size(), env_flag("WTIDE_GENERIC"));
  const int B = (int)g->pad_pot.size();
  *out = std::string("chain: ") + (p.plane_fast ? "k_plane_fast" : "k_plane") + " + " + (p.line_fast ? (env_flag("WTIDE_PENCIL1") ? "k_pencil" : "k_pencil2") : "k_spectral") +
         " + " + ((B > 640 || env_flag("WTIDE_SPLIT_BOUNDARY")) ? "k_boundary<1|2> + k_boundary_qh" : (p.plane_fast && g->nx == g->ny && g->nx != 96 ? "k_boundary_fast (cluster)" : "k_boundary_cluster")) +
         ", CUDA graph per output step";
}

int chain_solve(std::vector<GeomHost>& gs, GridDev gd, int* dstep, cudaStream_t st, SolveStats* stats) {
  const int n_geoms = (int)gs.size();
  const wt_geometry* g0 = gs[0].g;
  const int nx = g0->nx, ny = g0->ny, nz = g0->nz, y2 = ny / 2, nt = g0->nt;
  int maxB = 0, maxL = 0, maxG = 0, maxGL = 0, max_sub = 0;
  for (int i = 0; i < n_geoms; ++i) {
    maxB = std::max(maxB, (int)gs[i].g->pad_pot.size());
    maxL = std::max(maxL, (int)gs[i].g->layers.size());
    maxG = std::max(maxG, (int)gs[i].pg->grp_x.size());
    maxGL = std::max(maxGL, gs[i].pg->max_per_layer);
    max_sub = std::max(max_sub, gs[i].g->n_sub);
  }
  const Plan plan = make_plan(nx, ny, nz, maxL, env_flag("WTIDE_GENERIC"));
  const BndSmem bsm = bnd_smem(nx, ny, maxGL, maxB);
  const size_t kMaxSmem = 227 * 1024;
  const size_t sm_tr = (size_t)kStageSlots * 3 * std::max(nx, ny) * sizeof(float);
  const size_t sm_qh = ((size_t)2 * (nx / 2) * (ny + 1) + nx + ny) * sizeof(float2) + ((size_t)2 * nx + 2) * sizeof(int);     // k_boundary_qh: one layer image, two buffers
  // boundary adjust: one cluster launch per substep for small pad sets (16 CTAs where the device can
  // co-schedule the non-portable size, else 8), three grid-wide launches otherwise
  using BndFastFn = void (*)(const GeomBatch, GridDev, const BndClSmem, int, int, double);
  BndFastFn bnd_fast = nullptr;
  if (nx == ny && !env_flag("WTIDE_GENERIC")) {
    if (nx == 32) bnd_fast = k_boundary_fast<5, 4>;
    else if (nx == 64) bnd_fast = k_boundary_fast<6, 5>;
    else if (nx == 128) bnd_fast = k_boundary_fast<7, 6>;
  }
  const void* bnd_fn = bnd_fast ? (const void*)bnd_fast : (const void*)k_boundary_cluster<false>;
  const int bnd_threads = bnd_fast ? kBfThreads : kBclThreads;
  const int maxBs = (maxB + 1) & ~1;
  int bnd_cl = 8;
  BndClSmem bcl;
  int ainv_in_smem = 1;
  auto size_cluster = [&](int cl) {
    bnd_cl = cl; ainv_in_smem = 1;
    bcl = bnd_cl_smem(nx, ny, kMaxLayers, maxG, maxB, maxBs, cl, true, bnd_threads);
    if (bcl.total > 200 * 1024) { bcl = bnd_cl_smem(nx, ny, kMaxLayers, maxG, maxB, maxBs, cl, false, bnd_threads); ainv_in_smem = 0; }
  };
  size_cluster(16);
  bool bnd_cluster = maxB > 0 && maxB <= 640 && !env_flag("WTIDE_SPLIT_BOUNDARY");
  if (bnd_cluster) {
    bool ok16 = !env_flag("WTIDE_CLUSTER8") && bcl.total <= kMaxSmem &&
                cudaFuncSetAttribute(bnd_fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess &&
                cudaFuncSetAttribute(bnd_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bcl.total) == cudaSuccess;
    if (ok16) {
      cudaLaunchConfig_t q = {};
      q.gridDim = dim3(16, 1); q.blockDim = dim3(bnd_threads); q.dynamicSmemBytes = bcl.total;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = 16; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      q.attrs = at; q.numAttrs = 1;
      int n_clusters = 0;
      ok16 = cudaOccupancyMaxActiveClusters(&n_clusters, bnd_fn, &q) == cudaSuccess && n_clusters >= 1;
    }
    cudaGetLastError();
    if (!ok16) size_cluster(8);
    if (bcl.total > kMaxSmem) bnd_cluster = false;
  }
  if (plan.plane_smem > kMaxSmem || plan.line_smem > kMaxSmem || bsm.total > kMaxSmem || sm_tr > kMaxSmem || sm_qh > kMaxSmem) {
    wt_set_error("wt_solve_H: grid too large for the shared-memory tiles (nx*ny <= 128*128, nz <= 1024)"); return WT_EINVAL;
  }

  gd.ty = plan.ty; gd.n_tiles = nx * (y2 / plan.ty);
  gd.step = dstep;
#ifdef WTIDE_DEBUG
  gd.stamps = env_flag("WTIDE_STAMPS") ? (long long*)((char*)dstep + 256) : nullptr;
#endif
  CK(cudaMemsetAsync(dstep, 0, sizeof(int), st));
  // descriptors in launch batches of kBatch geometries
  const int n_batches = (n_geoms + kBatch - 1) / kBatch;
  std::vector<GeomBatch> batches(n_batches);
  std::vector<int> batch_n(n_batches);
  std::vector<GeomDev> hd(n_geoms);
  for (int i = 0; i < n_geoms; ++i) hd[i] = gs[i].dev;
  for (int bi = 0; bi < n_batches; ++bi) {
    batch_n[bi] = std::min(kBatch, n_geoms - bi * kBatch);
    for (int k = 0; k < kBatch; ++k) batches[bi].g[k] = hd[bi * kBatch + std::min(k, batch_n[bi] - 1)];
  }

  // ---- launch configuration -------------------------------------------------------------------
  auto set_smem = [&](const void* fn, size_t bytes) -> cudaError_t {
    return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  };
  CK(set_smem((const void*)plan.plane_step, plan.plane_smem)); CK(set_smem((const void*)plan.plane_emit, plan.plane_smem));
  CK(set_smem((const void*)plan.line_step, plan.line_smem)); CK(set_smem((const void*)plan.line_init, plan.line_smem));
  CK(set_smem((const void*)plan.line_delta, plan.line_smem));
  if (bnd_cluster) CK(set_smem(bnd_fn, bcl.total));
  CK(set_smem((const void*)k_boundary<1>, bsm.total));
  using QhFn = void (*)(const GeomBatch, GridDev, int);
  QhFn qh_fn = k_boundary_qh<0>;
  if (nx == ny && nx == 64) qh_fn = k_boundary_qh<64>;
  else if (nx == ny && nx == 96) qh_fn = k_boundary_qh<96>;
  else if (nx == ny && nx == 128) qh_fn = k_boundary_qh<128>;
  using B1Fn = void (*)(const GeomBatch, GridDev, int, int, int, double);
  B1Fn b1_fn = k_boundary<1>;
  if (nx == ny && nx == 64) b1_fn = k_boundary<1, 64>;
  else if (nx == ny && nx == 96) b1_fn = k_boundary<1, 96>;
  else if (nx == ny && nx == 128) b1_fn = k_boundary<1, 128>;
  CK(set_smem((const void*)b1_fn, bsm.total));
  CK(set_smem((const void*)k_boundary<2>, bsm.total)); CK(set_smem((const void*)qh_fn, sm_qh));
  CK(set_smem((const void*)k_transpose<false>, sm_tr)); CK(set_smem((const void*)k_transpose<true>, sm_tr));
  const int n_tr = plan.plane_fast ? nz * ny : nz * nx;
  const size_t half = (size_t)nx * nz * y2;
  const int bnd_rows = (maxB + kBndThreads / 32 - 1) / (kBndThreads / 32);

#ifdef WTIDE_DEBUG   // timing experiments only (drops kernels from the substep loop: WRONG results); never in the shipped library
  const int dbg_skip = std::getenv("WTIDE_DBG_SKIP") ? std::atoi(std::getenv("WTIDE_DBG_SKIP")) : 0;
#else
  constexpr int dbg_skip = 0;
#endif
  const bool pdl = !env_flag("WTIDE_NO_PDL");
  long long launches = 0;
  cudaError_t launch_err = cudaSuccess;
  auto note = [&](cudaError_t e) { if (e != cudaSuccess && launch_err == cudaSuccess) launch_err = e; };
  auto boundary = [&](int s, int emit, double flag) {
    if (maxB == 0) return;
    for (int bi = 0; bi < n_batches; ++bi) {
      const GeomBatch& gb = batches[bi];
      const int nb = batch_n[bi];
      if (bnd_cluster) {
        ++launches;
        if (bnd_fast) note(launch(bnd_fast, dim3(bnd_cl, nb), dim3(bnd_threads), bcl.total, st, pdl, bnd_cl, gb, gd, bcl, s, emit, flag));
        else note(launch(k_boundary_cluster<false>, dim3(bnd_cl, nb), dim3(bnd_threads), bcl.total, st, pdl, bnd_cl, gb, gd, maxG,
                         maxB, maxBs, ainv_in_smem, s, emit, flag));
      } else {
        launches += 3;
        note(launch(b1_fn, dim3(std::max(1, maxG), nb), dim3(kBndThreads), bsm.total, st, pdl, 1, gb, gd, maxGL, s, emit, flag));
        note(launch(k_boundary<2>, dim3(std::max(1, bnd_rows), nb), dim3(kBndThreads), bsm.total, st, pdl, 1, gb, gd, maxGL, s, emit, flag));
        note(launch(qh_fn, dim3(std::max(1, maxL), nb), dim3(kBndThreads), sm_qh, st, pdl, 1, gb, gd, s));
      }
    }
  };
  auto plane = [&](PlaneFn fn, int s) {
    for (int bi = 0; bi < n_batches; ++bi) {
      ++launches;
      const dim3 grid = plan.plane_fast ? dim3(nz, 3, batch_n[bi]) : dim3(nz, batch_n[bi]);
      note(launch(fn, grid, plan.plane_block, plan.plane_smem, st, pdl, 1, batches[bi], gd, s));
    }
  };
  auto line = [&](LineFn fn, int s, int emit) {
    for (int bi = 0; bi < n_batches; ++bi) {
      ++launches;
      note(launch(fn, dim3(plan.line_grid.x, batch_n[bi]), plan.line_block, plan.line_smem, st, pdl, 1, batches[bi], gd, s, emit));
    }
  };
  auto emit_step = [&](bool first) {
    // H[n] from the increment of the charge since the previous output step (the prompt response
    // H[0] from the pads alone: r = 0, pads at v_w); n is read from the device counter
    line(first ? plan.line_init : plan.line_delta, 0, 1);
    boundary(0, 1, first ? 1.0 : 0.0);
    plane(plan.plane_emit, 0);
    for (int bi = 0; bi < n_batches; ++bi) {
      ++launches;
      if (plan.plane_fast) note(launch(k_transpose<true>, dim3(n_tr, batch_n[bi]), dim3(256), sm_tr, st, pdl, 1, batches[bi], gd));
      else                 note(launch(k_transpose<false>, dim3(n_tr, batch_n[bi]), dim3(256), sm_tr, st, pdl, 1, batches[bi], gd));
    }
    ++launches;
    note(launch(k_advance, dim3(1), dim3(1), 0, st, pdl, 1, dstep));
  };
  auto output_step = [&]() {
    for (int s = 0; s < max_sub; ++s) {
      if (!(dbg_skip & 1)) boundary(s, 0, 1.0);
      if (!(dbg_skip & 2)) plane(plan.plane_step, s);
      if (!(dbg_skip & 4)) line(plan.line_step, s, 0);
    }
    emit_step(false);
  };

  for (int i = 0; i < n_geoms; ++i) {
    CK(cudaMemsetAsync(hd[i].rhat, 0, half * sizeof(double2), st));
    CK(cudaMemsetAsync(hd[i].rhat_prev, 0, half * sizeof(double2), st));
    if (hd[i].L > 0) CK(cudaMemsetAsync(hd[i].qh, 0, (size_t)hd[i].L * nx * y2 * sizeof(float2), st));
  }
  emit_step(true);
  line(plan.line_init, 0, 0);
  CK(cudaGetLastError());
  CK(launch_err);

  const int n_out = nt - 1;
  if (n_out >= 2 && !env_flag("WTIDE_NO_GRAPH")) {
    // one output step captured once, replayed n_out times
    const long long before = launches;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    CK(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
    output_step();
    cudaError_t ec = cudaStreamEndCapture(st, &graph);
    if (ec == cudaSuccess) ec = launch_err;
    if (ec != cudaSuccess || !graph) {
      if (graph) cudaGraphDestroy(graph);
      wt_set_error(std::string("wt_solve_H: stream capture failed: ") + cudaGetErrorString(ec)); return WT_ECUDA;
    }
    const long long per_step = launches - before;
    ec = cudaGraphInstantiate(&exec, graph, 0);
    if (ec != cudaSuccess) {
      cudaGraphDestroy(graph);
      wt_set_error(std::string("wt_solve_H: graph instantiation failed: ") + cudaGetErrorString(ec)); return WT_ECUDA;
    }
    for (int n = 0; n < n_out && ec == cudaSuccess; ++n) ec = cudaGraphLaunch(exec, st);
    launches = before + per_step * n_out;
    // an executable graph that is in flight is freed asynchronously on completion
    cudaGraphExecDestroy(exec);
    cudaGraphDestroy(graph);
    if (ec != cudaSuccess) { wt_set_error(std::string("wt_solve_H: graph launch failed: ") + cudaGetErrorString(ec)); return WT_ECUDA; }
  } else {
    for (int n = 0; n < n_out; ++n) output_step();
  }
  CK(cudaGetLastError());
  CK(launch_err);
  stats->launches += launches;
  return WT_OK;
}

}  // namespace wt
