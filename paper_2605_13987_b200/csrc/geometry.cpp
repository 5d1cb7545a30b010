// wt_make_geometry: step a0 of the hot path -- host setup in fp64.
//
// PAPER.md:64-65 ("the STL geometry is voxelized"), :95 (|k|^2), :97 (fundamental solution, point
// charges at the boundaries "adjusted, in magnitude, to enforce the boundary conditions").
// Readings R5-R13 of DESIGN.md.  The library works in units where eps = 1: r = rho/eps,
// s = sigma/eps [1/ns]; boundary charges Q' = Q/(eps*voxel volume).  H does not depend on that choice.
#include "geometry.h"

#include <algorithm>
#include <cmath>
#include <cstring>

static thread_local std::string g_err;
std::atomic<long long> g_wt_launches{0};
extern "C" int64_t wt_launch_count(void) { return (int64_t)g_wt_launches.load(); }
void wt_set_error(const std::string& msg) { g_err = msg; }
extern "C" const char* wt_last_error(void) { return g_err.c_str(); }
bool wt_valid(const wt_geometry* g) { return g != nullptr && g->magic == WT_MAGIC; }

bool wt_is_2a3b(int n) {
  if (n < 1) return false;
  while (n % 2 == 0) n /= 2;
  while (n % 3 == 0) n /= 3;
  return n == 1;
}

namespace {
const double kPi = 3.14159265358979323846;
// eps0 = 8.8541878128e-12 F/m in e/(V um); conductivity in e/(V um ns)  (same expressions as the
// descriptor's documentation so that the automatic substep count is reproducible by a caller)
const double kEps0 = 8.8541878128e-12 * 1e-6 / 1.602176634e-19;
double conductivity(double resistivity_ohm_cm) {
  return (1.0 / (resistivity_ohm_cm * 1e-2)) * 1e-6 * 1e-9 / 1.602176634e-19;
}

// signed mode number of DFT index k; the Nyquist index of an even n is flagged as removed (R11)
inline int mode_of(int k, int n, bool* removed) {
  *removed = (n % 2 == 0 && k == n / 2);
  return (2 * k < n) ? k : k - n;
}

// Inverse of a dense matrix by LU with partial pivoting (Doolittle), fp64.  Returns false if singular.
bool invert(std::vector<double>& a, int n, std::vector<double>& inv) {
  std::vector<int> piv(n);
  for (int i = 0; i < n; ++i) piv[i] = i;
  for (int c = 0; c < n; ++c) {
    int p = c;
    double best = std::fabs(a[(size_t)c * n + c]);
    for (int r = c + 1; r < n; ++r) {
      double v = std::fabs(a[(size_t)r * n + c]);
      if (v > best) { best = v; p = r; }
    }
    if (best == 0.0) return false;
    if (p != c) {
      for (int j = 0; j < n; ++j) std::swap(a[(size_t)p * n + j], a[(size_t)c * n + j]);
      std::swap(piv[p], piv[c]);
    }
    double d = 1.0 / a[(size_t)c * n + c];
    for (int r = c + 1; r < n; ++r) {
      double f = a[(size_t)r * n + c] * d;
      a[(size_t)r * n + c] = f;
      if (f != 0.0)
        for (int j = c + 1; j < n; ++j) a[(size_t)r * n + j] -= f * a[(size_t)c * n + j];
    }
  }
  inv.assign((size_t)n * n, 0.0);
  std::vector<double> col(n);
  for (int e = 0; e < n; ++e) {
    for (int i = 0; i < n; ++i) col[i] = (piv[i] == e) ? 1.0 : 0.0;
    for (int i = 0; i < n; ++i) {          // L y = P e
      double s = col[i];
      for (int j = 0; j < i; ++j) s -= a[(size_t)i * n + j] * col[j];
      col[i] = s;
    }
    for (int i = n - 1; i >= 0; --i) {     // U x = y
      double s = col[i];
      for (int j = i + 1; j < n; ++j) s -= a[(size_t)i * n + j] * col[j];
      col[i] = s / a[(size_t)i * n + i];
    }
    for (int i = 0; i < n; ++i) inv[(size_t)i * n + e] = col[i];
  }
  return true;
}
}  // namespace

extern "C" int wt_make_geometry(const wt_geometry_desc* d, wt_geometry** out) {
  if (!d || !out) { wt_set_error("wt_make_geometry: null argument"); return WT_EINVAL; }
  if (!(d->lx > 0 && d->ly > 0 && d->lz > 0 && d->dt > 0 && d->eps_r > 0 && d->v_w != 0)) {
    wt_set_error("wt_make_geometry: lx, ly, lz, dt, eps_r must be > 0 and v_w != 0"); return WT_EINVAL;
  }
  const int dims[3] = {d->nx, d->ny, d->nz};
  for (int a = 0; a < 3; ++a)
    if (dims[a] < 4 || dims[a] > 1024 || dims[a] % 2 != 0 || !wt_is_2a3b(dims[a])) {
      wt_set_error("wt_make_geometry: each grid size must be even, 2^a 3^b, 4 <= n <= 1024"); return WT_EINVAL;
    }
  if (d->nt < 4 || d->nt % 4 != 0) { wt_set_error("wt_make_geometry: nt must be a positive multiple of 4"); return WT_EINVAL; }
  if (d->n_columns < 1 || d->n_columns > 127 || !d->columns) {
    wt_set_error("wt_make_geometry: need 1..127 columns"); return WT_EINVAL;
  }
  if (d->substeps < 0) { wt_set_error("wt_make_geometry: substeps < 0"); return WT_EINVAL; }
  bool any_readout = false;
  for (int j = 0; j < d->n_columns; ++j) {
    const wt_column& c = d->columns[j];
    if (!(c.radius > 0 && c.resistivity > 0 && c.z0 >= 0 && c.z0 < c.z1 && c.z1 <= d->lz) ||
        (c.role != WT_BIAS && c.role != WT_READOUT) || !std::isfinite(c.cx) || !std::isfinite(c.cy)) {
      wt_set_error("wt_make_geometry: bad column " + std::to_string(j)); return WT_EINVAL;
    }
    any_readout |= (c.role == WT_READOUT);
  }
  if (!any_readout) { wt_set_error("wt_make_geometry: no readout column"); return WT_EGEOM; }

  wt_geometry* g = new wt_geometry();
  g->lx = d->lx; g->ly = d->ly; g->lz = d->lz;
  g->nx = d->nx; g->ny = d->ny; g->nz = d->nz; g->nt = d->nt;
  g->dt = d->dt; g->eps_r = d->eps_r; g->v_w = d->v_w; g->n_columns = d->n_columns;
  const int nx = g->nx, ny = g->ny, nz = g->nz, y2 = ny / 2;
  const size_t N = (size_t)nx * ny * nz;
  const double eps = d->eps_r * kEps0;

  // ---- voxeliser (R13): node-centre test, minimum image in x and y, first column wins ----------
  g->col_id.assign(N, (int8_t)-1);
  g->col_s.resize(d->n_columns);
  std::vector<double> xs(nx), ys(ny), zs(nz);
  for (int i = 0; i < nx; ++i) xs[i] = ((double)i * d->lx) / nx;
  for (int i = 0; i < ny; ++i) ys[i] = ((double)i * d->ly) / ny;
  for (int i = 0; i < nz; ++i) zs[i] = ((double)i * d->lz) / nz;
  double sigma_max = 0.0;
  for (int j = 0; j < d->n_columns; ++j) {
    const wt_column& c = d->columns[j];
    const double sig = conductivity(c.resistivity);
    g->col_s[j] = sig / eps;
    sigma_max = std::max(sigma_max, sig);
    int kfirst = -1, klast = -1;
    for (int k = 0; k < nz; ++k)
      if (c.z0 <= zs[k] && zs[k] <= c.z1) { if (kfirst < 0) kfirst = k; klast = k; }
    if (kfirst < 0) { delete g; wt_set_error("wt_make_geometry: column " + std::to_string(j) + " contains no grid node"); return WT_EGEOM; }
    const int kpad = c.pad_at_z1 ? klast : kfirst;
    const double r2 = c.radius * c.radius;
    bool any_xy = false;
    int n_pad = 0;
    for (int ix = 0; ix < nx; ++ix) {
      double dx = std::fmod(std::fabs(xs[ix] - c.cx), d->lx);
      dx = std::min(dx, d->lx - dx);
      for (int iy = 0; iy < ny; ++iy) {
        double dy = std::fmod(std::fabs(ys[iy] - c.cy), d->ly);
        dy = std::min(dy, d->ly - dy);
        if (!(dx * dx + dy * dy <= r2)) continue;
        any_xy = true;
        for (int k = 0; k < nz; ++k) {
          if (!(c.z0 <= zs[k] && zs[k] <= c.z1)) continue;
          int8_t& id = g->col_id[((size_t)ix * ny + iy) * nz + k];
          if (id >= 0) continue;
          id = (int8_t)j;
          ++g->n_conducting;
          if (k == kpad) {
            g->pad_nodes.push_back(ix); g->pad_nodes.push_back(iy); g->pad_nodes.push_back(k);
            g->pad_pot.push_back(c.role == WT_READOUT ? d->v_w : 0.0);
            ++n_pad;
          }
        }
      }
    }
    if (!any_xy) { delete g; wt_set_error("wt_make_geometry: column " + std::to_string(j) + " contains no grid node"); return WT_EGEOM; }
    if (n_pad == 0) { delete g; wt_set_error("wt_make_geometry: column " + std::to_string(j) + " has no pad node"); return WT_EGEOM; }
  }
  const int B = (int)g->pad_pot.size();

  // ---- substeps (R12) ----------------------------------------------------------------------------
  if (d->substeps == 0) {
    g->n_sub = std::max(1, (int)std::ceil(d->dt * (sigma_max / eps)));
  } else {
    g->n_sub = d->substeps;
    if (d->dt / d->substeps >= 2.0 * eps / sigma_max) {
      delete g; wt_set_error("wt_make_geometry: dt/substeps >= 2 eps/sigma_max, forward Euler is unstable"); return WT_EUNSTABLE;
    }
  }
  const double dt_int = d->dt / g->n_sub;

  // ---- pad layers ----------------------------------------------------------------------------------
  g->pad_layer.resize(B);
  for (int b = 0; b < B; ++b) {
    int k = g->pad_nodes[3 * b + 2];
    auto it = std::find(g->layers.begin(), g->layers.end(), k);
    if (it == g->layers.end()) { g->layers.push_back(k); it = g->layers.end() - 1; }
    g->pad_layer[b] = (int)(it - g->layers.begin());
  }
  const int L = (int)g->layers.size();

  // ---- conductivity map for the device: [z][x][y] ids and s*dt_int per id -------------------------
  g->sig_id.assign(N, 0);
  for (int ix = 0; ix < nx; ++ix)
    for (int iy = 0; iy < ny; ++iy)
      for (int k = 0; k < nz; ++k) {
        int8_t id = g->col_id[((size_t)ix * ny + iy) * nz + k];
        g->sig_id[((size_t)k * nx + ix) * ny + iy] = (uint8_t)(id + 1);
      }
  g->sdt.assign(256, 0.0f);
  for (int j = 0; j < d->n_columns; ++j) g->sdt[j + 1] = (float)(g->col_s[j] * dt_int);

  // ---- wavenumbers (step 1; Nyquist removed, R11) ---------------------------------------------------
  g->kx.resize(nx); g->ky.resize(y2); g->kz.resize(nz);
  std::vector<char> rx(nx), rz(nz);
  for (int k = 0; k < nx; ++k) { bool rm; int m = mode_of(k, nx, &rm); g->kx[k] = rm ? 0.0 : 2.0 * kPi * m / d->lx; rx[k] = !rm; }
  for (int k = 0; k < y2; ++k) g->ky[k] = 2.0 * kPi * k / d->ly;
  for (int k = 0; k < nz; ++k) { bool rm; int m = mode_of(k, nz, &rm); g->kz[k] = rm ? 0.0 : 2.0 * kPi * m / d->lz; rz[k] = !rm; }

  // ---- mixed-space fundamental solution (R9): for every retained (kx, ky >= 0)
  //   gt (kx,ky,dz) = sum_kz cos(2 pi m_z dz/nz) / |kappa|^2
  //   gzt(kx,ky,dz) = sum_kz kappa_z sin(2 pi m_z dz/nz) / |kappa|^2     (= -d/dz of gt)
  // over retained kz with (kx,ky,kz) != 0.  Layout [kx][dz][ky].
  g->gt.assign((size_t)nx * nz * y2, 0.0f);
  g->gzt.assign((size_t)nx * nz * y2, 0.0f);
  std::vector<double> gt64((size_t)nx * nz * y2, 0.0);   // kept in fp64 for the collocation matrix
  std::vector<double> cs(nz), sn(nz);
  for (int i = 0; i < nz; ++i) { cs[i] = std::cos(2.0 * kPi * i / nz); sn[i] = std::sin(2.0 * kPi * i / nz); }
  std::vector<double> w(nz);
  for (int ikx = 0; ikx < nx; ++ikx) {
    if (!rx[ikx]) continue;
    for (int iky = 0; iky < y2; ++iky) {
      const double kxy2 = g->kx[ikx] * g->kx[ikx] + g->ky[iky] * g->ky[iky];
      for (int ikz = 0; ikz < nz; ++ikz) {
        double k2 = kxy2 + g->kz[ikz] * g->kz[ikz];
        w[ikz] = (rz[ikz] && k2 > 0.0) ? 1.0 / k2 : 0.0;
      }
      for (int dz = 0; dz < nz; ++dz) {
        double a = 0.0, b = 0.0;
        for (int ikz = 0; ikz < nz; ++ikz) {
          if (w[ikz] == 0.0) continue;
          int ph = (int)(((int64_t)ikz * dz) % nz);        // e^{i kappa_z z}: index k and mode m give the same phase
          a += w[ikz] * cs[ph];
          b += w[ikz] * g->kz[ikz] * sn[ph];
        }
        size_t o = ((size_t)ikx * nz + dz) * y2 + iky;
        gt64[o] = a;
        g->gt[o] = (float)a;
        g->gzt[o] = (float)b;
      }
    }
  }

  // ---- bordered collocation matrix (step 4; R10) in eps = 1 units -----------------------------------
  //   G'(d) = (1/N) sum_k e^{i kappa.d}/|kappa|^2 = (1/N) sum_kx cos(kx dx) [gt(kx,0,dz) + 2 sum_{ky>0} cos(ky dy) gt(kx,ky,dz)]
  g->ainv.clear();
  if (B > 0) {
    std::vector<double> cx(nx), cy(ny);
    for (int i = 0; i < nx; ++i) cx[i] = std::cos(2.0 * kPi * i / nx);
    for (int i = 0; i < ny; ++i) cy[i] = std::cos(2.0 * kPi * i / ny);
    // planes of G' for every needed dz = (z_l - z_l') mod nz
    std::vector<int> dz_list;
    for (int a = 0; a < L; ++a)
      for (int b = 0; b < L; ++b) {
        int dz = ((g->layers[a] - g->layers[b]) % nz + nz) % nz;
        if (std::find(dz_list.begin(), dz_list.end(), dz) == dz_list.end()) dz_list.push_back(dz);
      }
    std::vector<std::vector<double>> planes(dz_list.size(), std::vector<double>((size_t)nx * ny));
    std::vector<double> t((size_t)nx * ny);
    for (size_t p = 0; p < dz_list.size(); ++p) {
      const int dz = dz_list[p];
      for (int ikx = 0; ikx < nx; ++ikx)
        for (int dy = 0; dy < ny; ++dy) {
          double s = gt64[((size_t)ikx * nz + dz) * y2 + 0];
          for (int iky = 1; iky < y2; ++iky) s += 2.0 * cy[(int)(((int64_t)iky * dy) % ny)] * gt64[((size_t)ikx * nz + dz) * y2 + iky];
          t[(size_t)ikx * ny + dy] = s;
        }
      for (int dx = 0; dx < nx; ++dx)
        for (int dy = 0; dy < ny; ++dy) {
          double s = 0.0;
          for (int ikx = 0; ikx < nx; ++ikx) s += cx[(int)(((int64_t)ikx * dx) % nx)] * t[(size_t)ikx * ny + dy];
          planes[p][(size_t)dx * ny + dy] = s / (double)N;
        }
    }
    const int n = B + 1;
    std::vector<double> a((size_t)n * n, 0.0), inv;
    for (int i = 0; i < B; ++i) {
      for (int j = 0; j < B; ++j) {
        int ddx = ((g->pad_nodes[3 * i] - g->pad_nodes[3 * j]) % nx + nx) % nx;
        int ddy = ((g->pad_nodes[3 * i + 1] - g->pad_nodes[3 * j + 1]) % ny + ny) % ny;
        int ddz = ((g->pad_nodes[3 * i + 2] - g->pad_nodes[3 * j + 2]) % nz + nz) % nz;
        size_t p = std::find(dz_list.begin(), dz_list.end(), ddz) - dz_list.begin();
        a[(size_t)i * n + j] = planes[p][(size_t)ddx * ny + ddy];
      }
      a[(size_t)i * n + B] = 1.0;
      a[(size_t)B * n + i] = 1.0;
    }
    if (!invert(a, n, inv)) { delete g; wt_set_error("wt_make_geometry: singular collocation matrix"); return WT_EGEOM; }
    g->ainv.resize((size_t)B * B);
    for (int i = 0; i < B; ++i)
      for (int j = 0; j < B; ++j) g->ainv[(size_t)i * B + j] = inv[(size_t)i * n + j];
  }
  *out = g;
  wt_set_error("");
  return WT_OK;
}

extern "C" void wt_free(void* handle) {
  wt_geometry* g = (wt_geometry*)handle;
  if (!g) return;
  if (g->magic != WT_MAGIC) return;
  g->magic = 0;
  delete g;
}

extern "C" int wt_get_array(const wt_geometry* g, int what, void* host_out, size_t bytes) {
  if (!wt_valid(g) || !host_out) { wt_set_error("wt_get_array: bad handle or null output"); return WT_EINVAL; }
  const void* src = nullptr;
  size_t need = 0;
  switch (what) {
    case WT_A_COLUMN_ID: src = g->col_id.data(); need = g->col_id.size(); break;
    case WT_A_PAD_NODES: src = g->pad_nodes.data(); need = g->pad_nodes.size() * sizeof(int32_t); break;
    case WT_A_PAD_POTENTIAL: src = g->pad_pot.data(); need = g->pad_pot.size() * sizeof(double); break;
    default: wt_set_error("wt_get_array: unknown array"); return WT_EINVAL;
  }
  if (bytes != need) { wt_set_error("wt_get_array: size mismatch, need " + std::to_string(need)); return WT_EINVAL; }
  std::memcpy(host_out, src, need);
  return WT_OK;
}
