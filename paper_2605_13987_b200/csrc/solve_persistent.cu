// Host side of the persistent solver (solve_persistent.cuh): kernel selection, grid / shared-memory sizing
// and the nt cooperative launches of one geometry's solve.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <string>

#include "solve_persistent.cuh"
#include "solve_plan.h"

namespace wt {
namespace {

constexpr int kMaxPadsPersistent = 1100;     // beyond: the kernel chain (Ainv streamed by the whole chip)

struct Variant {
  const void* fn;
  int tyl, pg, zg, max_pads;
  bool res;                 // one tile per z-line group, state resident in shared memory
  size_t phase_bytes, state_bytes;
};

template <int N, int EP, int NZ, int EZ, int TYL, bool RES>
Variant variant(int L) {
  using CF = PersistCfg<N, EP, NZ, EZ, TYL>;
  Variant v;
  v.fn = (L <= 2) ? (const void*)k_persistent<N, EP, NZ, EZ, TYL, 2, RES> : (const void*)k_persistent<N, EP, NZ, EZ, TYL, kMaxLayers, RES>;
  v.tyl = TYL; v.pg = CF::PG; v.zg = CF::ZG; v.res = RES;
  v.max_pads = ZGroupSmem<NZ, EZ, TYL>::max_pads;
  v.phase_bytes = CF::phase_bytes;
  v.state_bytes = RES ? CF::state_bytes : 0;
  return v;
}

bool pick(int nx, int ny, int nz, int L, Variant* v) {
  if (nx != ny) return false;
  if (nx == 64 && nz == 256) { *v = variant<64, 8, 256, 16, 8, true>(L); return true; }       // BASELINE configs 1 and 3
  if (nx == 128 && nz == 256) { *v = variant<128, 16, 256, 16, 8, false>(L); return true; }   // config 2
  // (config 0, 32^3, stays on the kernel chain: 11.5 us per substep there against 21 us here -- at that size the
  //  boundary hand-over between the CTAs costs more than three kernel boundaries)
  return false;
}

struct Sizing {
  int n_sm = 0, n_z = 0, n_b = 0, ainv_in_smem = 0;
  size_t smem = 0, persist_off = 0;
  bool ok = false;
};

Sizing size_launch(const wt_geometry* g, int B, const Variant& v) {
  Sizing s;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return s; }
  int n_sm = 0, max_smem = 0, coop = 0;
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  if (const char* e = std::getenv("WTIDE_PERSIST_SMS")) n_sm = std::min(n_sm, std::max(2, std::atoi(e)));
  if (!coop || n_sm < 2) return s;
  const int nx = g->nx, ny = g->ny, nz = g->nz, y2 = ny / 2;
  const int n_tiles = nx * (y2 / v.tyl);
  const int nb_min = std::max(1, std::min(20, (B + 31) / 32));
  if (n_sm - nb_min < 1) return s;
  const int per = (n_tiles + (n_sm - nb_min) * v.zg - 1) / ((n_sm - nb_min) * v.zg);   // tiles per z-line group
  const int n_z = (n_tiles + per * v.zg - 1) / (per * v.zg);
  const int p_ctas = (nz * 3 + v.pg - 1) / v.pg;
  const int grid = std::min(n_sm, std::max(n_z + nb_min, p_ctas));
  s.n_sm = n_sm; s.n_z = n_z; s.n_b = grid - n_z;
  if (B > v.max_pads) return s;
  if (v.res && (per != 1 || n_z * v.zg < n_tiles)) return s;      // (RES kernels own exactly one tile per group)
  const PersistSmem so = persist_smem(nx, ny, nz, B, v.res ? 0 : v.zg);
  s.persist_off = (so.phase + v.phase_bytes + 15) / 16 * 16;
  const int rows_per = (B + s.n_b - 1) / s.n_b, Bs = (B + 1) & ~1;
  const size_t bvec = (size_t)2 * Bs * 8, slice = (size_t)rows_per * Bs * 8;
  const size_t budget = (size_t)max_smem - 1024;      // (static shared memory of the kernel)
  const size_t need_min = s.persist_off + std::max(v.state_bytes, bvec);
  if (need_min > budget) return s;
  s.ainv_in_smem = (s.persist_off + bvec + slice <= budget && !env_flag("WTIDE_AINV_GLOBAL")) ? 1 : 0;
  s.smem = s.persist_off + std::max(v.state_bytes, bvec + (s.ainv_in_smem ? slice : 0));
  s.ok = true;
  return s;
}

}  // namespace

bool persistent_eligible(const wt_geometry* g, int n_pads) {
  Variant v;
  if (n_pads < 1 || n_pads > kMaxPadsPersistent || !pick(g->nx, g->ny, g->nz, (int)g->layers.size(), &v)) return false;
  return size_launch(g, n_pads, v).ok;
}

void persistent_describe(const wt_geometry* g, std::string* out) {
  Variant v;
  pick(g->nx, g->ny, g->nz, (int)g->layers.size(), &v);
  const Sizing s = size_launch(g, (int)g->pad_pot.size(), v);
  char buf[256];
  std::snprintf(buf, sizeof buf, "persistent: k_persistent<%d,%d> (plane_unit + z_pass_a/b + boundary CTAs), %d z-line + %d boundary CTAs, "
                "one cooperative launch per output step, state %s, Ainv %s", g->nx, g->nz, s.n_z, s.n_b,
                v.res ? "in shared memory" : "in L2", s.ainv_in_smem ? "in shared memory" : "from L2");
  *out = buf;
}

#define CKP(call)                                                                                   \
  do {                                                                                              \
    cudaError_t e_ = (call);                                                                        \
    if (e_ != cudaSuccess) {                                                                        \
      wt_set_error(std::string("wt_solve_H (persistent): ") + cudaGetErrorString(e_) + " at " #call); \
      return WT_ECUDA;                                                                              \
    }                                                                                               \
  } while (0)

int persistent_solve(GeomHost& gh, GridDev gd, cudaStream_t st, SolveStats* stats) {
  const wt_geometry* g = gh.g;
  const int B = (int)g->pad_pot.size(), L = (int)g->layers.size();
  Variant v;
  if (!pick(g->nx, g->ny, g->nz, (int)g->layers.size(), &v)) { wt_set_error("wt_solve_H (persistent): no kernel for this grid"); return WT_EINVAL; }
  const Sizing sz = size_launch(g, B, v);
  if (!sz.ok) { wt_set_error("wt_solve_H (persistent): launch does not fit the device"); return WT_ECUDA; }
  CKP(cudaFuncSetAttribute(v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sz.smem));
  int per_sm = 0;
  CKP(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, v.fn, kPersistThreads, sz.smem));
  if (per_sm < 1) { wt_set_error("wt_solve_H (persistent): kernel does not fit an SM"); return WT_ECUDA; }

  const size_t half = (size_t)g->nx * g->nz * (g->ny / 2);
  PersistArgs a = {};
  a.g = gh.dev; a.gd = gd;
  a.ctl = (PersistCtl*)(gh.base + gh.lo.ctl);
  a.fix = (long long*)(gh.base + gh.lo.part);
  a.pad_x = (const int*)(gh.base + gh.lo.pad_x);
  a.pad_l = (const int*)(gh.base + gh.lo.pad_l);
  for (int l = 0; l <= kMaxLayers; ++l) a.lpoff[l] = gh.pg->layer_poff[std::min(l, L)];
  a.n_z_cta = sz.n_z; a.n_b_cta = sz.n_b;
  a.ainv_in_smem = sz.ainv_in_smem; a.smem_persist_off = (unsigned)sz.persist_off;
#ifdef WTIDE_DEBUG
  a.stamps = env_flag("WTIDE_STAMPS") ? (unsigned long long*)(gh.base + gh.lo.dbg) : nullptr;
#endif
  CKP(cudaMemsetAsync(a.ctl, 0, sizeof(PersistCtl), st));
  CKP(cudaMemsetAsync(a.fix, 0, (size_t)2 * gh.dev.Bs * sizeof(long long), st));
  CKP(cudaMemsetAsync(gh.dev.rhat, 0, half * sizeof(double2), st));
  CKP(cudaMemsetAsync(gh.dev.rhat_prev, 0, half * sizeof(double2), st));

  const int nt = g->nt, n_sub = g->n_sub;
  unsigned long long bar = 0, epi = 0;
  for (int n = 0; n < nt; ++n) {
    a.step = n; a.n_sub = (n == 0) ? 0 : n_sub;
    a.bar0 = bar; a.epi0 = epi;
    void* kargs[] = {(void*)&a};
    CKP(cudaLaunchCooperativeKernel(v.fn, dim3(sz.n_z + sz.n_b), dim3(kPersistThreads), kargs, sz.smem, st));
    const bool tr = ((n + 1) % kStageSlots == 0) || n == nt - 1;
    bar += (n == 0 ? 1 : 2 * (unsigned long long)n_sub + 1) + (tr ? 1 : 0);
    epi += (n == 0 ? 1 : (unsigned long long)n_sub + 1);
    ++stats->launches;
  }
  k_persist_finish<<<1, 1, 0, st>>>(a.ctl, gh.dev.H);
  ++stats->launches;
  CKP(cudaGetLastError());
  return WT_OK;
}

}  // namespace wt
