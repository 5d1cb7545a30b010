// Internal host-side geometry object of libwtide (not part of the ABI).
#pragma once
#include <atomic>
#include <cstdint>
#include <memory>
#include <string>
#include <vector>

#include "../../include/wtide.h"

#define WT_MAGIC 0x57544744u /* "WTGD" */

struct wt_geometry {
  uint32_t magic = WT_MAGIC;
  // descriptor
  double lx, ly, lz;
  int nx, ny, nz, nt;
  double dt, eps_r, v_w;
  int n_sub;
  int n_columns;
  // setup results (host, fp64)
  std::vector<int8_t> col_id;       // [nx][ny][nz], -1 = diamond
  std::vector<double> col_s;        // per column: s = sigma/eps in 1/ns
  std::vector<float> cols_f32;      // per column: (float)cx, (float)cy, (float)r * (float)r  (transport kernels, next.cu)
  std::vector<int32_t> pad_nodes;   // [B][3]
  std::vector<double> pad_pot;      // [B]
  std::vector<int32_t> layers;      // distinct pad z-layers
  std::vector<int32_t> pad_layer;   // [B] index into layers
  int64_t n_conducting = 0;
  // tables uploaded by wt_solve_H (see solve.cu for their use)
  std::vector<uint8_t> sig_id;      // [z][x][y]: 0 = diamond, j+1 = column j
  std::vector<float> sdt;           // [256]: s * dt_int of id
  std::vector<float> gt, gzt;       // [kx][dz][ky] mixed-space fundamental solution and its -d/dz
  std::vector<double> ainv;         // [B][B] upper-left block of the inverse bordered matrix
  std::vector<double> kx, ky, kz;   // wavenumbers (0 at the removed Nyquist index); ky has ny/2 entries
  std::shared_ptr<void> solve_cache;   // what wt_solve_H derives from the handle on its first call (solve.cu: SolveCache)
};

extern std::atomic<long long> g_wt_launches;   // kernels launched by this process (wt_launch_count)
void wt_set_error(const std::string& msg);
bool wt_valid(const wt_geometry* g);
bool wt_is_2a3b(int n);
bool wt_build_solve_cache(wt_geometry* g);   // solve.cu: what wt_solve_H uploads, packed once per handle (host only)
