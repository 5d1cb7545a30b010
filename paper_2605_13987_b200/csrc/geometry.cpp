// wt_make_geometry: step a0 of the hot path -- host setup in fp64.
//
// PAPER.md:64-65 ("the STL geometry is voxelized"), :95 (|k|^2), :97 (fundamental solution, point
// charges at the boundaries "adjusted, in magnitude, to enforce the boundary conditions").
// Readings R5-R13 of DESIGN.md.  The library works in units where eps = 1: r = rho/eps,
// s = sigma/eps [1/ns]; boundary charges Q' = Q/(eps*voxel volume).  H does not depend on that choice.
#include "geometry.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdlib>
#include <cstring>
#include <thread>

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

// Runs fn(t, n_threads) on n_threads host threads (t = 0 runs on the caller).
template <typename F>
void parallel_run(int n_threads, F fn) {
  if (n_threads <= 1) { fn(0, 1); return; }
  std::vector<std::thread> th;
  th.reserve(n_threads - 1);
  for (int t = 1; t < n_threads; ++t) th.emplace_back([&fn, t, n_threads] { fn(t, n_threads); });
  fn(0, n_threads);
  for (auto& x : th) x.join();
}

int host_threads(size_t work) {
  if (work < (size_t)1 << 22) return 1;
  unsigned hc = std::thread::hardware_concurrency();
  if (hc == 0) hc = 1;
  if (const char* e = std::getenv("WTIDE_HOST_THREADS")) hc = (unsigned)std::max(1, std::atoi(e));
  return (int)std::min(hc, 32u);
}

// c[0..n) -= f * r[0..n): the inner loop of the elimination (contiguous, vectorised per ISA at load time)
__attribute__((target_clones("arch=skylake-avx512", "arch=haswell", "default")))
void row_axpy4(double* __restrict__ c, const double* __restrict__ r0, const double* __restrict__ r1, const double* __restrict__ r2,
               const double* __restrict__ r3, double f0, double f1, double f2, double f3, int n) {
  for (int j = 0; j < n; ++j) c[j] -= f0 * r0[j] + f1 * r1[j] + f2 * r2[j] + f3 * r3[j];
}
// the same for two rows c, d at once (the four pivot rows are loaded once for both)
__attribute__((target_clones("arch=skylake-avx512", "arch=haswell", "default")))
void row_axpy4x2(double* __restrict__ c, double* __restrict__ d, const double* __restrict__ r0, const double* __restrict__ r1,
                 const double* __restrict__ r2, const double* __restrict__ r3, const double* __restrict__ f, const double* __restrict__ h, int n) {
  const double f0 = f[0], f1 = f[1], f2 = f[2], f3 = f[3], h0 = h[0], h1 = h[1], h2 = h[2], h3 = h[3];
  for (int j = 0; j < n; ++j) {
    const double a0 = r0[j], a1 = r1[j], a2 = r2[j], a3 = r3[j];
    c[j] -= f0 * a0 + f1 * a1 + f2 * a2 + f3 * a3;
    d[j] -= h0 * a0 + h1 * a1 + h2 * a2 + h3 * a3;
  }
}

// In-place inverse of a symmetric positive definite matrix (row-major, n x n) by blocked Gauss-Jordan
// elimination without pivoting (stable for SPD matrices: it is the elimination order of an LDL^T
// factorisation), the rank-NB updates of the other rows spread over the host threads.
// Returns false if a pivot is not positive (matrix not numerically SPD).
bool invert_spd(std::vector<double>& a, int n) {
  constexpr int NB = 64;
  const int n_thr = host_threads((size_t)n * n * n / 8);
  std::vector<double> rowblk((size_t)NB * n), dinv((size_t)NB * NB), colblk((size_t)n * NB);
  for (int k0 = 0; k0 < n; k0 += NB) {
    const int nb = std::min(NB, n - k0);
    // invert the diagonal block (unblocked Gauss-Jordan, no pivoting)
    for (int i = 0; i < nb; ++i)
      for (int j = 0; j < nb; ++j) dinv[i * NB + j] = a[(size_t)(k0 + i) * n + k0 + j];
    for (int c = 0; c < nb; ++c) {
      const double piv = dinv[c * NB + c];
      if (!(piv > 0.0) || !std::isfinite(piv)) return false;
      const double d = 1.0 / piv;
      dinv[c * NB + c] = 1.0;
      for (int j = 0; j < nb; ++j) dinv[c * NB + j] *= d;
      for (int r = 0; r < nb; ++r) {
        if (r == c) continue;
        const double f = dinv[r * NB + c];
        dinv[r * NB + c] = 0.0;
        for (int j = 0; j < nb; ++j) dinv[r * NB + j] -= f * dinv[c * NB + j];
      }
    }
    // pivot rows R = D^-1 A[k,:] with the block column replaced by D^-1; keep the old block column of all rows
    parallel_run(std::min(n_thr, nb), [&](int t, int nt_) {
      for (int i = t; i < nb; i += nt_) {
        double* out = &rowblk[(size_t)i * n];
        for (int j = 0; j < n; ++j) out[j] = 0.0;
        for (int p = 0; p < nb; ++p) {
          const double f = dinv[i * NB + p];
          const double* src = &a[(size_t)(k0 + p) * n];
          for (int j = 0; j < n; ++j) out[j] += f * src[j];
        }
        for (int j = 0; j < nb; ++j) out[k0 + j] = dinv[i * NB + j];
      }
    });
    for (int r = 0; r < n; ++r)
      for (int p = 0; p < nb; ++p) { colblk[(size_t)r * NB + p] = a[(size_t)r * n + k0 + p]; }
    // every other row: A[r,:] -= A[r,k] R, with its block column set to -A[r,k] D^-1
    parallel_run(n_thr, [&](int t, int nt_) {
      auto one_row = [&](int r) {
        double* c = &a[(size_t)r * n];
        const double* f = &colblk[(size_t)r * NB];
        for (int p = 0; p < nb; ++p) c[k0 + p] = 0.0;
        int p = 0;
        for (; p + 3 < nb; p += 4)
          row_axpy4(c, &rowblk[(size_t)p * n], &rowblk[(size_t)(p + 1) * n], &rowblk[(size_t)(p + 2) * n], &rowblk[(size_t)(p + 3) * n],
                    f[p], f[p + 1], f[p + 2], f[p + 3], n);
        for (; p < nb; ++p) {
          const double fp = f[p];
          const double* rr = &rowblk[(size_t)p * n];
          for (int j = 0; j < n; ++j) c[j] -= fp * rr[j];
        }
      };
      // rows in pairs (2 t, 2 t + 1), (2 t + 2 nt_, ...): a pair that touches the pivot block falls back to single rows
      for (int r = 2 * t; r < n; r += 2 * nt_) {
        const int r2 = r + 1;
        const bool in0 = (r >= k0 && r < k0 + nb), in1 = (r2 >= n) || (r2 >= k0 && r2 < k0 + nb);
        if (in0 || in1 || nb % 4 != 0) {
          if (!in0) one_row(r);
          if (r2 < n && !(r2 >= k0 && r2 < k0 + nb)) one_row(r2);
          continue;
        }
        double* c = &a[(size_t)r * n];
        double* d = &a[(size_t)r2 * n];
        const double* f = &colblk[(size_t)r * NB];
        const double* h = &colblk[(size_t)r2 * NB];
        for (int p = 0; p < nb; ++p) { c[k0 + p] = 0.0; d[k0 + p] = 0.0; }
        for (int p = 0; p < nb; p += 4)
          row_axpy4x2(c, d, &rowblk[(size_t)p * n], &rowblk[(size_t)(p + 1) * n], &rowblk[(size_t)(p + 2) * n],
                      &rowblk[(size_t)(p + 3) * n], f + p, h + p, n);
      }
    });
    for (int i = 0; i < nb; ++i) std::memcpy(&a[(size_t)(k0 + i) * n], &rowblk[(size_t)i * n], (size_t)n * sizeof(double));
  }
  return true;
}

// In-place complex DFT of length n = 2^a 3^b (fp64, e^{+2 pi i jk/n}), recursive decimation in time with a
// twiddle table tw[k] = e^{+2 pi i k/n_top}; `stride` = n_top / n.  Used for the z-sums of the fundamental solution.
void dft_rec(std::complex<double>* x, std::complex<double>* tmp, int n, int stride, const std::complex<double>* tw) {
  if (n == 1) return;
  const int r = (n % 2 == 0) ? 2 : 3, m = n / r;
  // split into r interleaved subsequences, transform each
  for (int q = 0; q < r; ++q)
    for (int j = 0; j < m; ++j) tmp[q * m + j] = x[j * r + q];
  for (int q = 0; q < r; ++q) dft_rec(tmp + q * m, x, m, stride * r, tw);   // (x serves as scratch)
  if (r == 2) {
    for (int k = 0; k < m; ++k) {
      const std::complex<double> e = tmp[k], o = tmp[m + k] * tw[(size_t)k * stride];
      x[k] = e + o; x[k + m] = e - o;
    }
  } else {
    const std::complex<double> w3 = tw[(size_t)m * stride], w32 = tw[(size_t)2 * m * stride];   // e^{2 pi i/3}, e^{4 pi i/3}
    for (int k = 0; k < m; ++k) {
      const std::complex<double> a0 = tmp[k], a1 = tmp[m + k] * tw[(size_t)k * stride], a2 = tmp[2 * m + k] * tw[(size_t)2 * k * stride];
      x[k] = a0 + a1 + a2;
      x[k + m] = a0 + w3 * a1 + w32 * a2;
      x[k + 2 * m] = a0 + w32 * a1 + w3 * a2;
    }
  }
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
  if (d->mirror_z) {
    // Mirror (Neumann) surfaces at z = 0 and z = lz by the method of images: the even extension of the
    // sensor about both planes is periodic with period 2 lz, so the periodic solver runs on the doubled box
    if (d->mirror_z != 1 || 2 * d->nz > 1024 || 2 * d->n_columns > 127) {
      wt_set_error("wt_make_geometry: mirror_z must be 0 or 1 and needs 2 nz <= 1024, 2 n_columns <= 127"); return WT_EINVAL;
    }
    wt_geometry_desc m = *d;
    m.mirror_z = 0; m.lz = 2.0 * d->lz; m.nz = 2 * d->nz; m.n_columns = 2 * d->n_columns;
    std::vector<wt_column> cols(d->columns, d->columns + d->n_columns);
    for (int j = 0; j < d->n_columns; ++j) {
      const wt_column& c = d->columns[j];
      if (!(c.z0 >= 0 && c.z0 < c.z1 && c.z1 <= d->lz)) { wt_set_error("wt_make_geometry: bad column " + std::to_string(j)); return WT_EINVAL; }
      int kfirst = -1, klast = -1;               // the column's layers on the doubled grid, as the voxeliser finds them
      for (int k = 0; k < m.nz; ++k) {
        const double z = ((double)k * m.lz) / m.nz;
        if (c.z0 <= z && z <= c.z1) { if (kfirst < 0) kfirst = k; klast = k; }
      }
      const int kpad = c.pad_at_z1 ? klast : kfirst;
      wt_column im = c;
      im.z0 = m.lz - c.z1; im.z1 = m.lz - c.z0;
      im.pad_at_z1 = c.pad_at_z1 ? 0 : 1;
      if (c.role != WT_SEGMENT && (kpad == 0 || kpad == d->nz)) im.role = WT_SEGMENT;   // the pad is its own image
      cols.push_back(im);
    }
    m.columns = cols.data();
    return wt_make_geometry(&m, out);
  }
  bool any_readout = false;
  for (int j = 0; j < d->n_columns; ++j) {
    const wt_column& c = d->columns[j];
    if (!(c.radius > 0 && c.resistivity > 0 && c.z0 >= 0 && c.z0 < c.z1 && c.z1 <= d->lz) ||
        (c.role != WT_BIAS && c.role != WT_READOUT && c.role != WT_SEGMENT) || !std::isfinite(c.cx) || !std::isfinite(c.cy)) {
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
    g->cols_f32.push_back((float)c.cx); g->cols_f32.push_back((float)c.cy); g->cols_f32.push_back((float)c.radius * (float)c.radius);
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
          if (k == kpad && c.role != WT_SEGMENT) {
            g->pad_nodes.push_back(ix); g->pad_nodes.push_back(iy); g->pad_nodes.push_back(k);
            g->pad_pot.push_back(c.role == WT_READOUT ? d->v_w : 0.0);
            ++n_pad;
          }
        }
      }
    }
    if (!any_xy) { delete g; wt_set_error("wt_make_geometry: column " + std::to_string(j) + " contains no grid node"); return WT_EGEOM; }
    if (n_pad == 0 && c.role != WT_SEGMENT) { delete g; wt_set_error("wt_make_geometry: column " + std::to_string(j) + " has no pad node"); return WT_EGEOM; }
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
  // Per (kx, ky) these are the real and imaginary part of ONE length-nz DFT of the real sequence w + w kappa_z
  // (w = 1/|kappa|^2 is even in kz, w kappa_z is odd), O(N log nz) in total instead of O(N nz); lines over host threads.
  g->gt.assign((size_t)nx * nz * y2, 0.0f);
  g->gzt.assign((size_t)nx * nz * y2, 0.0f);
  std::vector<double> gt64((size_t)nx * nz * y2, 0.0);   // kept in fp64 for the collocation matrix
  {
    std::vector<std::complex<double>> tw(nz);
    for (int i = 0; i < nz; ++i) tw[i] = std::complex<double>(std::cos(2.0 * kPi * i / nz), std::sin(2.0 * kPi * i / nz));
    parallel_run(host_threads(N * 8), [&](int t, int nt_) {
      std::vector<std::complex<double>> line(nz), tmp(nz);
      for (int ikx = t; ikx < nx; ikx += nt_) {
        if (!rx[ikx]) continue;
        for (int iky = 0; iky < y2; ++iky) {
          const double kxy2 = g->kx[ikx] * g->kx[ikx] + g->ky[iky] * g->ky[iky];
          for (int ikz = 0; ikz < nz; ++ikz) {
            const double k2 = kxy2 + g->kz[ikz] * g->kz[ikz];
            const double w = (rz[ikz] && k2 > 0.0) ? 1.0 / k2 : 0.0;
            line[ikz] = std::complex<double>(w + w * g->kz[ikz], 0.0);
          }
          dft_rec(line.data(), tmp.data(), nz, 1, tw.data());
          for (int dz = 0; dz < nz; ++dz) {
            const size_t o = ((size_t)ikx * nz + dz) * y2 + iky;
            gt64[o] = line[dz].real();
            g->gt[o] = (float)line[dz].real();
            g->gzt[o] = (float)line[dz].imag();
          }
        }
      }
    });
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
    // Upper-left B x B block of the inverse of [[G,1],[1^T,0]] by the Schur complement of the SPD Green block:
    //   Ainv_BB = G^-1 - u u^T / (1^T u),  u = G^-1 1       (the constant c is never used, R33)
    std::vector<double> a((size_t)B * B);
    for (int i = 0; i < B; ++i)
      for (int j = 0; j < B; ++j) {
        int ddx = ((g->pad_nodes[3 * i] - g->pad_nodes[3 * j]) % nx + nx) % nx;
        int ddy = ((g->pad_nodes[3 * i + 1] - g->pad_nodes[3 * j + 1]) % ny + ny) % ny;
        int ddz = ((g->pad_nodes[3 * i + 2] - g->pad_nodes[3 * j + 2]) % nz + nz) % nz;
        size_t p = std::find(dz_list.begin(), dz_list.end(), ddz) - dz_list.begin();
        a[(size_t)i * B + j] = planes[p][(size_t)ddx * ny + ddy];
      }
    if (!invert_spd(a, B)) { delete g; wt_set_error("wt_make_geometry: singular collocation matrix (Green block not positive definite)"); return WT_EGEOM; }
    std::vector<double> u(B, 0.0);
    double ssum = 0.0;
    for (int i = 0; i < B; ++i) {
      double s = 0.0;
      for (int j = 0; j < B; ++j) s += a[(size_t)i * B + j];
      u[i] = s; ssum += s;
    }
    if (!(ssum != 0.0) || !std::isfinite(ssum)) { delete g; wt_set_error("wt_make_geometry: singular collocation matrix"); return WT_EGEOM; }
    g->ainv.resize((size_t)B * B);
    for (int i = 0; i < B; ++i) {
      const double ui = u[i] / ssum;
      for (int j = 0; j < B; ++j) g->ainv[(size_t)i * B + j] = a[(size_t)i * B + j] - ui * u[j];
    }
  }
  if (!wt_build_solve_cache(g)) { delete g; wt_set_error("wt_make_geometry: out of host memory"); return WT_ENOMEM; }
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
    case WT_A_AINV: src = g->ainv.data(); need = g->ainv.size() * sizeof(double); break;
    case WT_A_GT: src = g->gt.data(); need = g->gt.size() * sizeof(float); break;
    case WT_A_GZT: src = g->gzt.data(); need = g->gzt.size() * sizeof(float); break;
    default: wt_set_error("wt_get_array: unknown array"); return WT_EINVAL;
  }
  if (bytes != need) { wt_set_error("wt_get_array: size mismatch, need " + std::to_string(need)); return WT_EINVAL; }
  std::memcpy(host_out, src, need);
  return WT_OK;
}
