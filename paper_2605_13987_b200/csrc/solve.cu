// wt_solve_H: steps a1-a8 of the hot path on one B200 (sm_100a) -- argument checks, static tables, dispatch.
//
// Method (Fig. 3 :109; readings R1-R20 of DESIGN.md): forward Euler on
//   r <- r - dt_int div_s( s E ),  E = -grad_s V,  V = (r + boundary charges)/|kappa|^2 ,
// in units eps = 1 (r = rho/eps, s = sigma/eps).  The 3-D DFT is split into z-line transforms
// (tiles of z-lines (kx, few ky)) and xy-plane transforms (one plane z at a time); the fields between them
// live in "mixed space" arrays M[kx][z][ky] (ky >= 0 half spectrum).  One Euler substep =
//   boundary   pad potentials of the free charge -> rhs; Q' = Ainv rhs: "adjusted, in magnitude, to enforce
//              the boundary conditions" (a3); the translated fundamental solutions of the charges (a4)
//   plane      E~ = -i kappa V~; inverse xy DFT (a5); J = s dt_int E (a6); forward xy DFT; i kx J~x, i ky J~y, J~z
//   z-line     forward z DFT; r^ -= D^ + i kz J^z (a7, fp64 state); V^ = r^/|kappa|^2 (a2); inverse z DFT
// and every n_sub substeps the same phases run once on the increment r^ - r^_prev with the pads at 0 V and
// write H[n] = E/dt (a8) through a staging buffer that turns the time-innermost table writes into 96-byte runs.
//
// Two executions of these phases exist (solve_plan.h): the persistent kernel (one cooperative launch per
// output step, solve_persistent.cu) for the power-of-two grids of the BASELINE configs, and the kernel chain
// (one kernel per phase, CUDA graph, solve_chain.cu) for everything else.  A batch is split between them per
// geometry.  The static tables of a geometry are packed once per handle (by wt_make_geometry) into one host blob and
// reach the workspace with a single copy per call.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <string>
#include <utility>
#include <vector>

#include "solve_plan.h"

namespace wt {

bool env_flag(const char* name) {
  const char* v = std::getenv(name);
  return v && v[0] && v[0] != '0';
}

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
  o.pad_y.resize(B); o.pad_x.resize(B); o.pad_l.resize(B); o.pad_pot.resize(B); o.ainv.assign((size_t)B * Bs, 0.0);
  o.layer_poff.assign(L + 1, 0);
  for (int i = 0; i < B; ++i) {
    o.pad_x[i] = g->pad_nodes[3 * o.perm[i]];
    o.pad_y[i] = g->pad_nodes[3 * o.perm[i] + 1];
    o.pad_l[i] = g->pad_layer[o.perm[i]];
    o.layer_poff[o.pad_l[i] + 1]++;
    o.pad_pot[i] = g->pad_pot[o.perm[i]];
    for (int k = 0; k < B; ++k) o.ainv[(size_t)i * Bs + k] = g->ainv[(size_t)o.perm[i] * B + o.perm[k]];
  }
  for (int l = 0; l < L; ++l) o.layer_poff[l + 1] += o.layer_poff[l];
  return o;
}

Layout make_layout(const wt_geometry* g) {
  Layout o;
  const size_t nx = g->nx, ny = g->ny, nz = g->nz, y2 = ny / 2;
  const size_t N = nx * ny * nz, half = nx * nz * y2;
  const size_t B = g->pad_pot.size(), L = g->layers.size();
  size_t p = 0;
  auto take = [&](size_t bytes) { size_t at = p; p = align_up(p + bytes); return at; };
  o.sig_id = take(N); o.sig_t = take(N); o.sdt = take(256 * 4); o.gt = take(half * 4); o.gzt = take(half * 4);
  o.ainv = take(B * ((B + 1) & ~(size_t)1) * 8); o.pad_pot = take(B * 8); o.pad_y = take(B * 4); o.pad_x = take(B * 4); o.pad_l = take(B * 4);
  o.grp_x = take(B * 4); o.grp_layer = take(B * 4); o.grp_off = take((B + 1) * 4);
  o.layer_goff = take((L + 1) * 4);
  o.kxd = take(nx * 8); o.kyd = take(y2 * 8); o.kzd = take(nz * 8);
  o.kxf = take(nx * 4); o.kyf = take(y2 * 4); o.kzf = take(nz * 4);
  o.twx = take(nx * 8); o.twy = take(ny * 8); o.twz = take(nz * 8);
  o.twxd = take(nx * 16); o.twyd = take(ny * 16); o.twzd = take(nz * 16);
  o.static_bytes = p;
  o.rhat = take(half * 16); o.rhat_prev = take(half * 16);
  o.v0 = take(half * 8); o.v1 = take(half * 8);
  o.m0 = take(half * 8); o.m1 = take(half * 8); o.m2 = take(half * 8); o.e0 = take(half * 8); o.e1 = take(half * 8);
  o.pl = take(L * nx * y2 * 16); o.pl_e = take(L * nx * y2 * 16);
  o.rhs = take(B * 8); o.q = take(B * 8); o.qh = take(L * nx * y2 * 8);
  o.part = take(((B + 1) & ~(size_t)1) * 2 * 8); o.ctl = take(256);   // (persistent kernel: int64 pad potentials, control block)
  o.stage = take((size_t)kStageSlots * 3 * N * 4);
#ifdef WTIDE_DEBUG
  o.dbg = take(256 * 1024);
#endif
  o.total = p;
  return o;
}

namespace {

// What wt_solve_H derives from a handle once and keeps on it: the pad groups, the workspace layout and the
// static section of the workspace as one pinned host blob.
struct SolveCache {
  PadGroups pg;
  Layout lo;
  char* blob = nullptr;        // pageable: packed by wt_make_geometry (host only), one cudaMemcpyAsync per wt_solve_H call
  ~SolveCache() { std::free(blob); }
};

template <typename T>
void put(char* blob, size_t off, const std::vector<T>& v) {
  if (!v.empty()) std::memcpy(blob + off, v.data(), v.size() * sizeof(T));
}

SolveCache* get_cache(wt_geometry* g) {
  if (g->solve_cache) return static_cast<SolveCache*>(g->solve_cache.get());
  auto c = std::make_shared<SolveCache>();
  c->pg = make_groups(g);
  c->lo = make_layout(g);
  const Layout& lo = c->lo;
  const PadGroups& pg = c->pg;
  c->blob = (char*)std::malloc(lo.static_bytes);
  if (!c->blob) return nullptr;
  std::memset(c->blob, 0, lo.static_bytes);
  char* b = c->blob;
  const int nx = g->nx, ny = g->ny, nz = g->nz;
  std::vector<uint8_t> sig_t(g->sig_id.size());
  for (int z = 0; z < nz; ++z)
    for (int x = 0; x < nx; ++x)
      for (int y = 0; y < ny; ++y) sig_t[((size_t)z * ny + y) * nx + x] = g->sig_id[((size_t)z * nx + x) * ny + y];
  std::vector<float> kxf(g->kx.begin(), g->kx.end()), kyf(g->ky.begin(), g->ky.end()), kzf(g->kz.begin(), g->kz.end());
  // twiddles e^{-2 pi i k/n} (fp64 on the host)
  const double kPi = 3.14159265358979323846;
  auto twid = [&](int n, std::vector<float2>& f, std::vector<double2>& d) {
    f.resize(n); d.resize(n);
    for (int k = 0; k < n; ++k) {
      const double cs = std::cos(2.0 * kPi * k / n), sn = -std::sin(2.0 * kPi * k / n);
      d[k] = make_double2(cs, sn); f[k] = make_float2((float)cs, (float)sn);
    }
  };
  std::vector<float2> twx, twy, twz;
  std::vector<double2> twxd, twyd, twzd;
  twid(nx, twx, twxd); twid(ny, twy, twyd); twid(nz, twz, twzd);
  put(b, lo.sig_id, g->sig_id); put(b, lo.sig_t, sig_t); put(b, lo.sdt, g->sdt);
  put(b, lo.gt, g->gt); put(b, lo.gzt, g->gzt);
  put(b, lo.ainv, pg.ainv); put(b, lo.pad_pot, pg.pad_pot); put(b, lo.pad_y, pg.pad_y); put(b, lo.pad_x, pg.pad_x); put(b, lo.pad_l, pg.pad_l);
  put(b, lo.grp_x, pg.grp_x); put(b, lo.grp_layer, pg.grp_layer); put(b, lo.grp_off, pg.grp_off); put(b, lo.layer_goff, pg.layer_goff);
  put(b, lo.kxd, g->kx); put(b, lo.kyd, g->ky); put(b, lo.kzd, g->kz);
  put(b, lo.kxf, kxf); put(b, lo.kyf, kyf); put(b, lo.kzf, kzf);
  put(b, lo.twx, twx); put(b, lo.twy, twy); put(b, lo.twz, twz);
  put(b, lo.twxd, twxd); put(b, lo.twyd, twyd); put(b, lo.twzd, twzd);
  g->solve_cache = c;
  return c.get();
}

bool use_persistent(const wt_geometry* g) {
  return !env_flag("WTIDE_CHAIN") && !env_flag("WTIDE_GENERIC") && persistent_eligible(g, (int)g->pad_pot.size());
}

#define CK(call)                                                                              \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      wt_set_error(std::string("wt_solve_H: ") + cudaGetErrorString(e_) + " at " #call);      \
      return WT_ECUDA;                                                                        \
    }                                                                                         \
  } while (0)

}  // namespace
}  // namespace wt

using namespace wt;

// called at the end of wt_make_geometry (host work, part of the setup a0): pad groups, layout, packed static tables
bool wt_build_solve_cache(wt_geometry* g) { return get_cache(g) != nullptr; }

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
  for (int i = 0; i < n_geoms; ++i) {
    const wt_geometry* g = geoms[i];
    if (!wt_valid(g) || !H_dev[i]) { wt_set_error("wt_solve_H: bad handle or null table pointer"); return WT_EINVAL; }
    if (g->nx != g0->nx || g->ny != g0->ny || g->nz != g0->nz || g->nt != g0->nt) {
      wt_set_error("wt_solve_H: all geometries of a batch must share grid and nt"); return WT_EINVAL;
    }
    if ((int)g->layers.size() > kMaxLayers) { wt_set_error("wt_solve_H: more than 8 distinct pad layers"); return WT_EINVAL; }
    if (((uintptr_t)H_dev[i]) % 16 != 0) { wt_set_error("wt_solve_H: H table not 16-byte aligned"); return WT_EINVAL; }
    regions += make_layout(g).total;
  }
  const size_t need = regions + 4096;
  const size_t hbytes = (size_t)g0->nx * g0->ny * g0->nz * g0->nt * 12;
  if (H_bytes_each < hbytes) { wt_set_error("wt_solve_H: H_bytes_each too small"); return WT_EINVAL; }
  if (((uintptr_t)workspace_dev) % 256 != 0) { wt_set_error("wt_solve_H: workspace not 256-byte aligned"); return WT_EINVAL; }
  if (workspace_bytes < need) { wt_set_error("wt_solve_H: workspace too small, need " + std::to_string(need)); return WT_ENOMEM; }

  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nx = g0->nx, ny = g0->ny, nz = g0->nz, y2 = ny / 2, nt = g0->nt;
  GridDev gd = {};
  gd.nx = nx; gd.ny = ny; gd.nz = nz; gd.y2 = y2; gd.nt = nt; gd.ty = 1; gd.n_tiles = 0;
  gd.inv_n = 1.0 / ((double)nx * ny * nz);

  // ---- static tables (one copy per geometry), descriptors (which travel as kernel parameters) -----------
  std::vector<GeomHost> all(n_geoms);
  char* base = (char*)workspace_dev;
  size_t off = 0;
  for (int i = 0; i < n_geoms; ++i) {
    wt_geometry* g = geoms[i];
    SolveCache* sc = get_cache(g);
    if (!sc) { wt_set_error("wt_solve_H: out of host memory for the static tables"); return WT_ENOMEM; }
    const Layout& lo = sc->lo;
    const PadGroups& pg = sc->pg;
    char* b = base + off;
    const int B = (int)g->pad_pot.size(), L = (int)g->layers.size();
    CK(cudaMemcpyAsync(b, sc->blob, lo.static_bytes, cudaMemcpyHostToDevice, st));
    GeomHost& gh = all[i];
    gh.g = g; gh.pg = &sc->pg; gh.lo = lo; gh.base = b;
    GeomDev& d = gh.dev;
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

  // ---- dispatch: persistent kernel per eligible geometry, the kernel chain for the rest (as one lock-step batch)
  SolveStats stats;
  std::vector<GeomHost> chain;
  for (int i = 0; i < n_geoms; ++i) {
    if (use_persistent(all[i].g)) {
      const int rc = persistent_solve(all[i], gd, st, &stats);
      if (rc != WT_OK) return rc;
    } else {
      chain.push_back(all[i]);
    }
  }
  if (!chain.empty()) {
    const int rc = chain_solve(chain, gd, dstep, st, &stats);
    if (rc != WT_OK) return rc;
  }
  g_wt_launches += stats.launches;
  wt_set_error("");
  return WT_OK;
}

#ifdef WTIDE_DEBUG
extern "C" int64_t wt_debug_stamps_offset(const wt_geometry* g) { return (int64_t)make_layout(g).dbg; }
#endif

extern "C" int wt_describe_plan(const wt_geometry* g, char* out, size_t out_bytes) {
  if (!wt_valid(g) || !out || out_bytes == 0) { wt_set_error("wt_describe_plan: bad argument"); return WT_EINVAL; }
  std::string s;
  if (use_persistent(g)) persistent_describe(g, &s);
  else chain_describe(g, &s);
  std::snprintf(out, out_bytes, "%s", s.c_str());
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
    case WT_Q_N_COLUMNS: *value = g->n_columns; break;
    case WT_Q_NZ: *value = g->nz; break;
    default: wt_set_error("wt_query: unknown item"); return WT_EINVAL;
  }
  return WT_OK;
}
