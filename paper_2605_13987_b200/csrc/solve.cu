// wt_solve_H: steps a1-a8 of the hot path on one B200 (sm_100a).
//
// Method (Fig. 3 :109; readings R1-R20 of DESIGN.md): forward Euler on
//   r <- r - dt_int div_s( s E ),  E = -grad_s V,  V = (r + boundary charges)/|kappa|^2 ,
// in units eps = 1 (r = rho/eps, s = sigma/eps).  The 3-D DFT is split into z-line transforms
// (one CTA per (kx, tile of ky)) and xy-plane transforms (one CTA per z); the fields between them
// live in "mixed space" arrays M[kx][z][ky] (ky >= 0 half spectrum).
//
// One Euler substep =
//   boundary   pad potentials of the free charge from pl = V~_rho at the pad layers -> rhs;           (a3)
//              Q' = Ainv rhs: "adjusted, in magnitude, to enforce the boundary conditions";          (a3)
//              spectrum of the boundary point charges per pad layer                                 (a4)
//              (one cluster launch, or three grid-wide launches for large pad sets)
//   plane      V~ = V~_rho + sum_l Q^_l * g~ (translated fundamental solution, a4); E~ = -i kappa V~;
//              inverse xy DFT (a5); J = s dt_int E (a6); forward xy DFT; i kx J~x, i ky J~y, J~z
//   z-line     forward z DFT; r^ -= D^ + i kz J^z (a7, fp64 state); V^ = r^/|kappa|^2 (a2);
//              pl (fp64); inverse z DFT of V^ and -i kz V^
// Every n_sub substeps the same kernels run once on the increment r^ - r^_prev with the pads at
// 0 V and write H[n] = E/dt (a8) through a staging buffer that turns the time-innermost table
// writes into 12*TB-byte runs (k_transpose).  The kernels of one output step (n_sub substeps + emit)
// are captured once into a CUDA graph and replayed nt-1 times; the output-step index lives in a
// device counter.  Plane and z-line kernels come in a size-generic family (solve_generic.cuh) and a
// register-FFT family for power-of-two sizes (solve_fast.cuh).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <string>
#include <utility>
#include <vector>

#include "geometry.h"
#include "solve_boundary.cuh"
#include "solve_fast.cuh"
#include "solve_generic.cuh"

namespace {
using namespace wt;

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

int pick_ty(int y2) {
  const int cand[6] = {8, 6, 4, 3, 2, 1};
  for (int c : cand)
    if (y2 % c == 0) return c;
  return 1;
}

bool env_flag(const char* name) {
  const char* v = std::getenv(name);
  return v && v[0] && v[0] != '0';
}

// pads of one geometry grouped by (layer, x); perm[i] = index (in the handle's pad order) of the
// i-th pad in group order; the device holds every per-pad array in group order
struct PadGroups {
  std::vector<int> grp_x, grp_layer, grp_off, perm, layer_goff, pad_y;
  std::vector<double> pad_pot, ainv;
  int max_per_layer = 0;
};

PadGroups make_groups(const wt_geometry* g) {
  PadGroups o;
  const int B = (int)g->pad_pot.size(), L = (int)g->layers.size();
  std::map<std::pair<int, int>, std::vector<int>> m;
  for (int b = 0; b < B; ++b) m[{g->pad_layer[b], g->pad_nodes[3 * b]}].push_back(b);
  o.layer_goff.assign(L + 1, 0);
  o.grp_off.push_back(0);
  for (auto& kv : m) {
    o.grp_layer.push_back(kv.first.first);
    o.grp_x.push_back(kv.first.second);
    for (int b : kv.second) o.perm.push_back(b);
    o.grp_off.push_back((int)o.perm.size());
    o.layer_goff[kv.first.first + 1]++;
  }
  for (int l = 0; l < L; ++l) {
    o.max_per_layer = std::max(o.max_per_layer, o.layer_goff[l + 1]);
    o.layer_goff[l + 1] += o.layer_goff[l];
  }
  const int Bs = (B + 1) & ~1;    // even row stride: rows and row slices start 16-byte aligned
  o.pad_y.resize(B); o.pad_pot.resize(B); o.ainv.assign((size_t)B * Bs, 0.0);
  for (int i = 0; i < B; ++i) {
    o.pad_y[i] = g->pad_nodes[3 * o.perm[i] + 1];
    o.pad_pot[i] = g->pad_pot[o.perm[i]];
    for (int k = 0; k < B; ++k) o.ainv[(size_t)i * Bs + k] = g->ainv[(size_t)o.perm[i] * B + o.perm[k]];
  }
  return o;
}

// Offsets of one geometry's region inside the workspace (static tables, then state).
struct Layout {
  size_t sig_id, sig_t, sdt, gt, gzt, ainv, pad_pot, pad_y, grp_x, grp_layer, grp_off, layer_goff;
  size_t kxd, kyd, kzd, kxf, kyf, kzf, twx, twy, twz, twxd, twyd, twzd;
  size_t rhat, rhat_prev, v0, v1, m0, m1, m2, e0, e1, pl, pl_e, rhs, q, qh, stage;
  size_t total;
};

Layout make_layout(const wt_geometry* g) {
  Layout o;
  const size_t nx = g->nx, ny = g->ny, nz = g->nz, y2 = ny / 2;
  const size_t N = nx * ny * nz, half = nx * nz * y2;
  const size_t B = g->pad_pot.size(), L = g->layers.size();
  size_t p = 0;
  auto take = [&](size_t bytes) { size_t at = p; p = align_up(p + bytes); return at; };
  o.sig_id = take(N); o.sig_t = take(N); o.sdt = take(256 * 4); o.gt = take(half * 4); o.gzt = take(half * 4);
  o.ainv = take(B * ((B + 1) & ~(size_t)1) * 8); o.pad_pot = take(B * 8); o.pad_y = take(B * 4);
  o.grp_x = take(B * 4); o.grp_layer = take(B * 4); o.grp_off = take((B + 1) * 4);
  o.layer_goff = take((L + 1) * 4);
  o.kxd = take(nx * 8); o.kyd = take(y2 * 8); o.kzd = take(nz * 8);
  o.kxf = take(nx * 4); o.kyf = take(y2 * 4); o.kzf = take(nz * 4);
  o.twx = take(nx * 8); o.twy = take(ny * 8); o.twz = take(nz * 8);
  o.twxd = take(nx * 16); o.twyd = take(ny * 16); o.twzd = take(nz * 16);
  o.rhat = take(half * 16); o.rhat_prev = take(half * 16);
  o.v0 = take(half * 8); o.v1 = take(half * 8);
  o.m0 = take(half * 8); o.m1 = take(half * 8); o.m2 = take(half * 8); o.e0 = take(half * 8); o.e1 = take(half * 8);
  o.pl = take(L * nx * y2 * 16); o.pl_e = take(L * nx * y2 * 16);
  o.rhs = take(B * 8); o.q = take(B * 8); o.qh = take(L * nx * y2 * 8);
  o.stage = take((size_t)kStageSlots * 3 * N * 4);
  o.total = p;
  return o;
}

template <typename T>
cudaError_t upload(char* base, size_t off, const std::vector<T>& v, cudaStream_t st) {
  if (v.empty()) return cudaSuccess;
  return cudaMemcpyAsync(base + off, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st);
}

#define CK(call)                                                                              \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      wt_set_error(std::string("wt_solve_H: ") + cudaGetErrorString(e_) + " at " #call);      \
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
    p.line_smem = (size_t)3 * nz * p.ty * sizeof(float2) + (size_t)std::max(1, L) * p.ty * 32 * sizeof(double2) + (size_t)nz * sizeof(float2);
  }
  return p;
}

}  // namespace

// bytes wt_solve_H needs for this geometry (its region + one descriptor slot + the step counter)
size_t wt_solve_workspace_bytes(const wt_geometry* g) { return make_layout(g).total + 4096; }

extern "C" int wt_solve_H(wt_geometry* const* geoms, int n_geoms, float* const* H_dev, size_t H_bytes_each,
                          void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  if (!geoms || n_geoms < 1 || !H_dev || !workspace_dev || !cuda_stream) {
    wt_set_error("wt_solve_H: null argument, n_geoms < 1 or NULL (default) stream"); return WT_EINVAL;
  }
  const wt_geometry* g0 = geoms[0];
  if (!wt_valid(g0)) { wt_set_error("wt_solve_H: bad handle"); return WT_EINVAL; }
  size_t regions = 0;
  int max_sub = 0;
  for (int i = 0; i < n_geoms; ++i) {
    const wt_geometry* g = geoms[i];
    if (!wt_valid(g) || !H_dev[i]) { wt_set_error("wt_solve_H: bad handle or null table pointer"); return WT_EINVAL; }
    if (g->nx != g0->nx || g->ny != g0->ny || g->nz != g0->nz || g->nt != g0->nt) {
      wt_set_error("wt_solve_H: all geometries of a batch must share grid and nt"); return WT_EINVAL;
    }
    if ((int)g->layers.size() > kMaxLayers) { wt_set_error("wt_solve_H: more than 8 distinct pad layers"); return WT_EINVAL; }
    if (((uintptr_t)H_dev[i]) % 16 != 0) { wt_set_error("wt_solve_H: H table not 16-byte aligned"); return WT_EINVAL; }
    regions += make_layout(g).total;
    max_sub = std::max(max_sub, g->n_sub);
  }
  const size_t need = regions + 4096;
  const size_t hbytes = (size_t)g0->nx * g0->ny * g0->nz * g0->nt * 12;
  if (H_bytes_each < hbytes) { wt_set_error("wt_solve_H: H_bytes_each too small"); return WT_EINVAL; }
  if (((uintptr_t)workspace_dev) % 256 != 0) { wt_set_error("wt_solve_H: workspace not 256-byte aligned"); return WT_EINVAL; }
  if (workspace_bytes < need) { wt_set_error("wt_solve_H: workspace too small, need " + std::to_string(need)); return WT_ENOMEM; }

  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nx = g0->nx, ny = g0->ny, nz = g0->nz, y2 = ny / 2, nt = g0->nt;
  int maxB = 0, maxL = 0, maxG = 0, maxGL = 0;
  std::vector<PadGroups> groups(n_geoms);
  for (int i = 0; i < n_geoms; ++i) {
    groups[i] = make_groups(geoms[i]);
    maxB = std::max(maxB, (int)geoms[i]->pad_pot.size());
    maxL = std::max(maxL, (int)geoms[i]->layers.size());
    maxG = std::max(maxG, (int)groups[i].grp_x.size());
    maxGL = std::max(maxGL, groups[i].max_per_layer);
  }
  const Plan plan = make_plan(nx, ny, nz, maxL, env_flag("WTIDE_GENERIC"));
  const BndSmem bsm = bnd_smem(nx, ny, maxGL, maxB);
  const size_t kMaxSmem = 227 * 1024;
  const size_t sm_tr = (size_t)kStageSlots * 3 * std::max(nx, ny) * sizeof(float);
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
  if (plan.plane_smem > kMaxSmem || plan.line_smem > kMaxSmem || bsm.total > kMaxSmem || sm_tr > kMaxSmem) {
    wt_set_error("wt_solve_H: grid too large for the shared-memory tiles (nx*ny <= 128*128, nz <= 1024)"); return WT_EINVAL;
  }

  GridDev gd;
  gd.nx = nx; gd.ny = ny; gd.nz = nz; gd.y2 = y2; gd.nt = nt; gd.ty = plan.ty; gd.n_tiles = nx * (y2 / plan.ty);
  gd.inv_n = 1.0 / ((double)nx * ny * nz);

  // twiddles e^{-2 pi i k/n} (fp64 on the host)
  const double kPi = 3.14159265358979323846;
  auto twid = [&](int n, std::vector<float2>& f, std::vector<double2>& d) {
    f.resize(n); d.resize(n);
    for (int k = 0; k < n; ++k) {
      const double c = std::cos(2.0 * kPi * k / n), s = -std::sin(2.0 * kPi * k / n);
      d[k] = make_double2(c, s); f[k] = make_float2((float)c, (float)s);
    }
  };
  std::vector<float2> twx, twy, twz;
  std::vector<double2> twxd, twyd, twzd;
  twid(nx, twx, twxd); twid(ny, twy, twyd); twid(nz, twz, twzd);

  // ---- upload static tables, build the descriptors (which travel as kernel parameters) -----------
  std::vector<GeomDev> hd(n_geoms);
  char* base = (char*)workspace_dev;
  size_t off = 0;
  std::vector<uint8_t> sig_t;
  std::vector<float> kxf, kyf, kzf;
  for (int i = 0; i < n_geoms; ++i) {
    const wt_geometry* g = geoms[i];
    const Layout lo = make_layout(g);
    const PadGroups& pg = groups[i];
    char* b = base + off;
    const int B = (int)g->pad_pot.size(), L = (int)g->layers.size();
    sig_t.resize(g->sig_id.size());
    for (int z = 0; z < nz; ++z)
      for (int x = 0; x < nx; ++x)
        for (int y = 0; y < ny; ++y) sig_t[((size_t)z * ny + y) * nx + x] = g->sig_id[((size_t)z * nx + x) * ny + y];
    kxf.assign(g->kx.begin(), g->kx.end()); kyf.assign(g->ky.begin(), g->ky.end()); kzf.assign(g->kz.begin(), g->kz.end());
    // (cudaMemcpyAsync from pageable memory has staged the source before it returns)
    CK(upload(b, lo.sig_id, g->sig_id, st)); CK(upload(b, lo.sig_t, sig_t, st)); CK(upload(b, lo.sdt, g->sdt, st));
    CK(upload(b, lo.gt, g->gt, st)); CK(upload(b, lo.gzt, g->gzt, st));
    CK(upload(b, lo.ainv, pg.ainv, st)); CK(upload(b, lo.pad_pot, pg.pad_pot, st)); CK(upload(b, lo.pad_y, pg.pad_y, st));
    CK(upload(b, lo.grp_x, pg.grp_x, st)); CK(upload(b, lo.grp_layer, pg.grp_layer, st));
    CK(upload(b, lo.grp_off, pg.grp_off, st)); CK(upload(b, lo.layer_goff, pg.layer_goff, st));
    CK(upload(b, lo.kxd, g->kx, st)); CK(upload(b, lo.kyd, g->ky, st)); CK(upload(b, lo.kzd, g->kz, st));
    CK(upload(b, lo.kxf, kxf, st)); CK(upload(b, lo.kyf, kyf, st)); CK(upload(b, lo.kzf, kzf, st));
    CK(upload(b, lo.twx, twx, st)); CK(upload(b, lo.twy, twy, st)); CK(upload(b, lo.twz, twz, st));
    CK(upload(b, lo.twxd, twxd, st)); CK(upload(b, lo.twyd, twyd, st)); CK(upload(b, lo.twzd, twzd, st));
    GeomDev& d = hd[i];
    d.sig_id = (const uint8_t*)(b + lo.sig_id); d.sig_t = (const uint8_t*)(b + lo.sig_t); d.sdt = (const float*)(b + lo.sdt);
    d.gt = (const float*)(b + lo.gt); d.gzt = (const float*)(b + lo.gzt);
    d.ainv = (const double*)(b + lo.ainv); d.pad_pot = (const double*)(b + lo.pad_pot); d.pad_y = (const int*)(b + lo.pad_y);
    d.grp_x = (const int*)(b + lo.grp_x); d.grp_layer = (const int*)(b + lo.grp_layer);
    d.grp_off = (const int*)(b + lo.grp_off); d.layer_goff = (const int*)(b + lo.layer_goff);
    d.kxd = (const double*)(b + lo.kxd); d.kyd = (const double*)(b + lo.kyd); d.kzd = (const double*)(b + lo.kzd);
    d.kxf = (const float*)(b + lo.kxf); d.kyf = (const float*)(b + lo.kyf); d.kzf = (const float*)(b + lo.kzf);
    d.twx = (const float2*)(b + lo.twx); d.twy = (const float2*)(b + lo.twy); d.twz = (const float2*)(b + lo.twz);
    d.twxd = (const double2*)(b + lo.twxd); d.twyd = (const double2*)(b + lo.twyd); d.twzd = (const double2*)(b + lo.twzd);
    d.rhat = (double2*)(b + lo.rhat); d.rhat_prev = (double2*)(b + lo.rhat_prev);
    d.v0 = (float2*)(b + lo.v0); d.v1 = (float2*)(b + lo.v1);
    d.m0 = (float2*)(b + lo.m0); d.m1 = (float2*)(b + lo.m1); d.m2 = (float2*)(b + lo.m2);
    d.e0 = (float2*)(b + lo.e0); d.e1 = (float2*)(b + lo.e1);
    d.pl = (double2*)(b + lo.pl); d.pl_e = (double2*)(b + lo.pl_e);
    d.rhs = (double*)(b + lo.rhs); d.q = (double*)(b + lo.q); d.qh = (float2*)(b + lo.qh);
    d.stage = (float*)(b + lo.stage);
    d.H = H_dev[i];
    for (int l = 0; l < kMaxLayers; ++l) d.layers[l] = (l < L) ? g->layers[l] : 0;
    for (int l = 0; l <= kMaxLayers; ++l) d.lgoff[l] = pg.layer_goff[std::min(l, L)];
    d.B = B; d.Bs = (B + 1) & ~1; d.L = L; d.G = (int)pg.grp_x.size(); d.n_sub = g->n_sub; d.inv_dt = (float)(1.0 / g->dt);
    off += lo.total;
  }
  int* dstep = (int*)(base + off);
  gd.step = dstep;
#ifdef WTIDE_DEBUG
  gd.stamps = env_flag("WTIDE_STAMPS") ? (long long*)(base + off + 256) : nullptr;
#endif
  CK(cudaMemsetAsync(dstep, 0, sizeof(int), st));
  // descriptors in launch batches of kBatch geometries
  const int n_batches = (n_geoms + kBatch - 1) / kBatch;
  std::vector<GeomBatch> batches(n_batches);
  std::vector<int> batch_n(n_batches);
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
  CK(set_smem((const void*)k_boundary<2>, bsm.total)); CK(set_smem((const void*)k_boundary<3>, bsm.total));
  CK(set_smem((const void*)k_transpose<false>, sm_tr)); CK(set_smem((const void*)k_transpose<true>, sm_tr));
  const int n_tr = plan.plane_fast ? nz * ny : nz * nx;
  const size_t half = (size_t)nx * nz * y2;
  const int bnd_units3 = std::max(1, maxL) * ((nx + kBndKx - 1) / kBndKx);
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
        note(launch(k_boundary<1>, dim3(std::max(1, maxG), nb), dim3(kBndThreads), bsm.total, st, pdl, 1, gb, gd, maxGL, s, emit, flag));
        note(launch(k_boundary<2>, dim3(std::max(1, bnd_rows), nb), dim3(kBndThreads), bsm.total, st, pdl, 1, gb, gd, maxGL, s, emit, flag));
        note(launch(k_boundary<3>, dim3(bnd_units3, nb), dim3(kBndThreads), bsm.total, st, pdl, 1, gb, gd, maxGL, s, emit, flag));
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
  g_wt_launches += launches;
  wt_set_error("");
  return WT_OK;
}

extern "C" int wt_query(const wt_geometry* g, int what, int64_t* value) {
  if (!wt_valid(g) || !value) { wt_set_error("wt_query: bad handle or null output"); return WT_EINVAL; }
  switch (what) {
    case WT_Q_H_BYTES: *value = (int64_t)g->nx * g->ny * g->nz * g->nt * 12; break;
    case WT_Q_SOLVE_WORKSPACE_BYTES: *value = (int64_t)wt_solve_workspace_bytes(g); break;
    case WT_Q_SUBSTEPS: *value = g->n_sub; break;
    case WT_Q_N_PADS: *value = (int64_t)g->pad_pot.size(); break;
    case WT_Q_N_NODES: *value = (int64_t)g->nx * g->ny * g->nz; break;
    case WT_Q_N_CONDUCTING: *value = g->n_conducting; break;
    case WT_Q_N_PAD_LAYERS: *value = (int64_t)g->layers.size(); break;
    case WT_Q_NT: *value = g->nt; break;
    default: wt_set_error("wt_query: unknown item"); return WT_EINVAL;
  }
  return WT_OK;
}
