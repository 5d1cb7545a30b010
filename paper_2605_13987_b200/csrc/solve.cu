// wt_solve_H: steps a1-a8 of the hot path on one B200 (sm_100a).
//
// Method (Fig. 3 :109; readings R1-R20 of DESIGN.md): forward Euler on
//   r <- r - dt_int div_s( s E ),  E = -grad_s V,  V = (r + boundary charges)/|kappa|^2 ,
// in units eps = 1 (r = rho/eps, s = sigma/eps).  The 3-D DFT is split into z-line transforms
// (k_spectral, one CTA per (kx, tile of ky)) and xy-plane transforms (k_plane, one CTA per z);
// the fields between them live in "mixed space" arrays M[kx][z][ky] (ky >= 0 half spectrum).
//
// One Euler substep =
//   k_rhs      pad potentials from the free charge (partials written by k_spectral) -> rhs      (a3)
//   k_matvec   Q' = Ainv rhs: "adjusted, in magnitude, to enforce the boundary conditions"       (a3)
//   k_inject   spectrum of the boundary point charges per pad layer                              (a4)
//   k_plane    V~ = V~_rho + sum_l Q^_l * g~ (translated fundamental solution, a4); E~ = -i kappa V~;
//              inverse xy DFT (a5); J = s dt_int E (a6); forward xy DFT; D~ = i kx J~x + i ky J~y
//   k_spectral forward z DFT; r^ -= D^ + i kz J^z (a7, fp64 state); V^ = r^/|kappa|^2 (a2);
//              pad-layer potentials (fp64); inverse z DFT of V^ and -i kz V^
// Every n_sub substeps the same kernels run once on the increment r^ - r^_prev with the pads at
// 0 V and write H[n] = E/dt (a8) through a staging buffer that turns the time-innermost table
// writes into 12*TB-byte runs (k_transpose).
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <string>
#include <vector>

#include "fft.cuh"
#include "geometry.h"

namespace {

constexpr int kMaxLayers = 8;
constexpr int kStageSlots = 8;   // TB: output steps buffered before a table write (96-byte runs)

struct GridDev {
  int nx, ny, nz, y2, nt, ty, n_tiles;   // n_tiles = nx * (y2/ty) = CTAs of k_spectral per geometry
  double inv_n;
};

struct GeomDev {
  // static tables
  const uint8_t* sig_id;     // [z][x][y]
  const float* sdt;          // [256]
  const float* gt;           // [kx][dz][ky]
  const float* gzt;
  const double* ainv;        // [B][B]
  const int* pad_x; const int* pad_y; const int* pad_layer;   // [B]
  const double* pad_pot;     // [B]
  const int* layer_off;      // [L+1] offsets into layer_idx
  const int* layer_idx;      // [B] pad indices grouped by layer
  const double* kxd; const double* kyd; const double* kzd;    // wavenumbers
  const float2* twx; const float2* twy; const float2* twz;    // e^{-2 pi i k/n}
  const double2* twxd; const double2* twyd; const double2* twzd;
  // state
  double2* rhat; double2* rhat_prev;   // [kx][kz][ky]
  float2* m0; float2* m1;              // step pipeline: (V~_rho | D~), (E~z_rho | J~z)   [kx][z][ky]
  float2* e0; float2* e1;              // emit pipeline
  double* part; double* part_e;        // [n_tiles][B] pad-potential partials
  double* rhs; double* q;              // [B]
  float2* qh;                          // [L][kx][ky] spectrum of the boundary charges
  float* stage;                        // [TB][3][z][x][y]
  float* H;
  int layers[kMaxLayers];
  int B, L, n_sub;
  float inv_dt;
};

__device__ __forceinline__ double2 dmul(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// ------------------------------------------------------------------------------------------------
// k_spectral: z-line transforms + per-mode update.  grid (n_tiles, n_geoms), block 32*ty.
// ------------------------------------------------------------------------------------------------
template <bool APPLY_J, bool DELTA>
__global__ void __launch_bounds__(256) k_spectral(GridDev gd, const GeomDev* __restrict__ geoms, int substep, int emit) {
  const GeomDev& g = geoms[blockIdx.y];
  if (substep >= g.n_sub) return;
  const int nx = gd.nx, nz = gd.nz, y2 = gd.y2, TY = gd.ty;
  const int tiles = y2 / TY;
  const int kx = blockIdx.x / tiles, ky0 = (blockIdx.x % tiles) * TY;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int nelem = nz * TY;
  const int L = g.L, B = g.B;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* b0 = reinterpret_cast<float2*>(smraw);
  float2* b1 = b0 + nelem;
  float2* b2 = b1 + nelem;
  double2* red = reinterpret_cast<double2*>(b2 + nelem);   // [L][TY][32]
  double2* pl = red + L * TY * 32;                          // [L][TY]
  float2* mV = emit ? g.e0 : g.m0;
  float2* mE = emit ? g.e1 : g.m1;
  const size_t slab = (size_t)kx * nz * y2 + ky0;

  float2 *dres, *jres, *vb;
  if (APPLY_J) {
    for (int t = tid; t < nelem; t += bd) {
      const int z = t / TY, ty = t - z * TY;
      const size_t gi = slab + (size_t)z * y2 + ty;
      b0[t] = g.m0[gi];
      b2[t] = g.m1[gi];
    }
    __syncthreads();
    dres = wt::fft_lines<float2>(b0, b1, nz, TY, 1, TY, g.twz, false);
    float2* free1 = (dres == b0) ? b1 : b0;
    jres = wt::fft_lines<float2>(b2, free1, nz, TY, 1, TY, g.twz, false);
    vb = (jres == b2) ? free1 : b2;
  } else {
    vb = b0; dres = b1; jres = b2;
  }

  // per-mode update (a7), potential from charge (a2), pad-layer partial sums (a3, fp64)
  double2 acc[kMaxLayers];
#pragma unroll
  for (int l = 0; l < kMaxLayers; ++l) acc[l] = make_double2(0.0, 0.0);
  const int ty = tid % TY;          // blockDim = 32*TY, so ty is fixed per thread
  const int ky = ky0 + ty;
  const double kxd = g.kxd[kx], kyd = g.kyd[ky];
  const bool ret_x = (kx != nx / 2);
  for (int t = tid; t < nelem; t += bd) {
    const int kz = t / TY;
    const size_t gi = ((size_t)kx * nz + kz) * y2 + ky;
    const bool ret = ret_x && (kz != nz / 2);
    const double kzd = g.kzd[kz];
    double2 r = g.rhat[gi];
    if (APPLY_J) {
      const float2 D = dres[t], J = jres[t];
      const float kzf = (float)kzd;
      r.x -= (double)(D.x - kzf * J.y);
      r.y -= (double)(D.y + kzf * J.x);
      if (!ret) r = make_double2(0.0, 0.0);
      g.rhat[gi] = r;
    }
    double2 src = r;
    if (DELTA) {
      const double2 p = g.rhat_prev[gi];
      src.x -= p.x; src.y -= p.y;
      g.rhat_prev[gi] = r;
    }
    const double k2 = kxd * kxd + kyd * kyd + kzd * kzd;
    const double gg = (ret && k2 > 0.0) ? gd.inv_n / k2 : 0.0;
    const double2 v = make_double2(src.x * gg, src.y * gg);
    vb[t] = make_float2((float)v.x, (float)v.y);
    dres[t] = make_float2((float)(kzd * v.y), (float)(-kzd * v.x));   // -i kz V^
#pragma unroll
    for (int l = 0; l < kMaxLayers; ++l) {
      if (l < L) {
        double2 w = g.twzd[(int)(((long long)kz * g.layers[l]) % nz)];
        w.y = -w.y;                                                    // e^{+i kz z_l}
        const double2 p = dmul(v, w);
        acc[l].x += p.x; acc[l].y += p.y;
      }
    }
  }
#pragma unroll
  for (int l = 0; l < kMaxLayers; ++l)
    if (l < L) red[(l * TY + ty) * 32 + tid / TY] = acc[l];
  __syncthreads();
  if (tid < L * TY) {
    double2 s = make_double2(0.0, 0.0);
    for (int i = 0; i < 32; ++i) { const double2 p = red[tid * 32 + i]; s.x += p.x; s.y += p.y; }
    pl[tid] = s;
  }
  __syncthreads();
  // contribution of this CTA's (kx, ky tile) modes to the potential at every pad node
  double* part = (emit ? g.part_e : g.part) + (size_t)blockIdx.x * B;
  for (int b = tid; b < B; b += bd) {
    const int l = g.pad_layer[b], x = g.pad_x[b], y = g.pad_y[b];
    double2 wx = g.twxd[(int)(((long long)kx * x) % nx)];
    wx.y = -wx.y;
    double val = 0.0;
    for (int j = 0; j < TY; ++j) {
      double2 wy = g.twyd[(int)(((long long)(ky0 + j) * y) % gd.ny)];
      wy.y = -wy.y;
      const double2 p = dmul(pl[l * TY + j], dmul(wx, wy));
      val += ((ky0 + j) == 0 ? 1.0 : 2.0) * p.x;
    }
    part[b] = val;
  }
  // inverse z transforms (a5, z part)
  float2* vres = wt::fft_lines<float2>(vb, jres, nz, TY, 1, TY, g.twz, true);
  float2* fr = (vres == vb) ? jres : vb;
  for (int t = tid; t < nelem; t += bd) {
    const int z = t / TY, tyy = t - z * TY;
    mV[slab + (size_t)z * y2 + tyy] = vres[t];
  }
  float2* eres = wt::fft_lines<float2>(dres, fr, nz, TY, 1, TY, g.twz, true);
  for (int t = tid; t < nelem; t += bd) {
    const int z = t / TY, tyy = t - z * TY;
    mE[slab + (size_t)z * y2 + tyy] = eres[t];
  }
}

// ------------------------------------------------------------------------------------------------
// boundary adjust (a3): rhs, Q' = Ainv rhs, spectrum of the point charges (a4)
// ------------------------------------------------------------------------------------------------
// one warp per pad: rhs[b] = flag*V_pad[b] - sum over tiles of the partial potentials (fixed order)
__global__ void __launch_bounds__(256) k_rhs(GridDev gd, const GeomDev* __restrict__ geoms, int substep, int emit, double flag) {
  const GeomDev& g = geoms[blockIdx.y];
  if (substep >= g.n_sub) return;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= g.B) return;
  const double* part = emit ? g.part_e : g.part;
  double s = 0.0;
  for (int c = lane; c < gd.n_tiles; c += 32) s += part[(size_t)c * g.B + warp];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) g.rhs[warp] = flag * g.pad_pot[warp] - s;
}

// one warp per row of Ainv
__global__ void __launch_bounds__(256) k_matvec(const GeomDev* __restrict__ geoms, int substep) {
  const GeomDev& g = geoms[blockIdx.y];
  if (substep >= g.n_sub) return;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= g.B) return;
  const double* row = g.ainv + (size_t)warp * g.B;
  double s = 0.0;
  for (int j = lane; j < g.B; j += 32) s += row[j] * g.rhs[j];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) g.q[warp] = s;
}

// one thread per (layer, kx, ky): Q^_l = (1/N) sum_{b in l} Q'_b e^{-i(kx x_b + ky y_b)}
__global__ void __launch_bounds__(256) k_inject(GridDev gd, const GeomDev* __restrict__ geoms, int substep) {
  const GeomDev& g = geoms[blockIdx.z];
  if (substep >= g.n_sub) return;
  const int l = blockIdx.y;
  if (l >= g.L) return;
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  const int nmodes = gd.nx * gd.y2;
  __shared__ int sx[256], sy[256];
  __shared__ double sq[256];
  const int kx = m / gd.y2, ky = m - kx * gd.y2;
  double2 acc = make_double2(0.0, 0.0);
  const int beg = g.layer_off[l], end = g.layer_off[l + 1];
  for (int c0 = beg; c0 < end; c0 += 256) {
    const int n = min(256, end - c0);
    __syncthreads();
    if ((int)threadIdx.x < n) {
      const int b = g.layer_idx[c0 + threadIdx.x];
      sx[threadIdx.x] = g.pad_x[b]; sy[threadIdx.x] = g.pad_y[b]; sq[threadIdx.x] = g.q[b];
    }
    __syncthreads();
    if (m < nmodes) {
      for (int i = 0; i < n; ++i) {
        const double2 w = dmul(g.twxd[(int)(((long long)kx * sx[i]) % gd.nx)], g.twyd[(int)(((long long)ky * sy[i]) % gd.ny)]);
        acc.x += sq[i] * w.x; acc.y += sq[i] * w.y;
      }
    }
  }
  if (m < nmodes) {
    if (kx == gd.nx / 2) acc = make_double2(0.0, 0.0);
    g.qh[(size_t)l * nmodes + m] = make_float2((float)(acc.x * gd.inv_n), (float)(acc.y * gd.inv_n));
  }
}

// ------------------------------------------------------------------------------------------------
// k_plane: xy-plane transforms.  grid (nz, n_geoms), block 256.
// Shared memory: three buffers of (nx/2)*(ny+1) float2 used either as a half-spectrum plane
// [kx][ky] (row stride y2) or as nx/2 complex lines of length ny, each packing the two real
// x-rows 2p (real part) and 2p+1 (imaginary part), line stride ny+1 (odd: conflict free).
// ------------------------------------------------------------------------------------------------
template <bool EMIT>
__global__ void __launch_bounds__(256) k_plane(GridDev gd, const GeomDev* __restrict__ geoms, int substep, int slot) {
  const GeomDev& g = geoms[blockIdx.y];
  if (substep >= g.n_sub) return;
  const int nx = gd.nx, ny = gd.ny, nz = gd.nz, y2 = gd.y2;
  const int z = blockIdx.x;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int nyp = ny + 1, hx = nx / 2;
  const int nspec = nx * y2, nline = hx * ny;
  const int bufsz = hx * nyp;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* dacc = reinterpret_cast<float2*>(smraw);
  float2* w1 = dacc + bufsz;
  float2* w2 = w1 + bufsz;
  const float2* mV = EMIT ? g.e0 : g.m0;
  const float2* mE = EMIT ? g.e1 : g.m1;
  const int L = g.L;

  for (int comp = 0; comp < 3; ++comp) {
    // (1) E~_comp on the half-spectrum plane, boundary-charge part added (a4)
    for (int t = tid; t < nspec; t += bd) {
      const int kx = t / y2, ky = t - kx * y2;
      const size_t gi = ((size_t)kx * nz + z) * y2 + ky;
      float2 v = (comp == 2) ? mE[gi] : mV[gi];
      const float* tab = (comp == 2) ? g.gzt : g.gt;
      for (int l = 0; l < L; ++l) {
        int dz = z - g.layers[l];
        if (dz < 0) dz += nz;
        const float gv = tab[((size_t)kx * nz + dz) * y2 + ky];
        const float2 qv = g.qh[(size_t)l * nspec + t];
        v.x += qv.x * gv; v.y += qv.y * gv;
      }
      if (comp < 2) {
        const float kap = (comp == 0) ? (float)g.kxd[kx] : (float)g.kyd[ky];
        v = make_float2(kap * v.y, -kap * v.x);               // -i kappa V~
      }
      w1[t] = v;
    }
    __syncthreads();
    // (2) inverse along x: y2 lines of length nx, element stride y2
    float2* r = wt::fft_lines<float2>(w1, w2, nx, y2, 1, y2, g.twx, true);
    float2* o = (r == w1) ? w2 : w1;
    // (3) pack two x-rows into one complex line with the Hermitian completion along y (Nyquist = 0)
    for (int t = tid; t < nline; t += bd) {
      const int p = t / ny, k = t - p * ny;
      float2 zv;
      if (k < y2) {
        const float2 a = r[(2 * p) * y2 + k], b = r[(2 * p + 1) * y2 + k];
        zv = make_float2(a.x - b.y, a.y + b.x);
      } else if (k == y2) {
        zv = make_float2(0.f, 0.f);
      } else {
        const float2 a = r[(2 * p) * y2 + (ny - k)], b = r[(2 * p + 1) * y2 + (ny - k)];
        zv = make_float2(a.x + b.y, b.x - a.y);
      }
      o[p * nyp + k] = zv;
    }
    __syncthreads();
    // (4) inverse along y: nx/2 lines of length ny
    float2* e = wt::fft_lines<float2>(o, r, ny, hx, nyp, 1, g.twy, true);
    float2* f = (e == o) ? r : o;
    if (EMIT) {
      // (a8) H[n] = E/dt into the staging slot, component-planar [slot][comp][z][x][y]
      float* st = g.stage + (((size_t)slot * 3 + comp) * nz + z) * (size_t)(nx * ny);
      for (int t = tid; t < nline; t += bd) {
        const int p = t / ny, y = t - p * ny;
        const float2 v = e[p * nyp + y];
        st[(2 * p) * ny + y] = v.x * g.inv_dt;
        st[(2 * p + 1) * ny + y] = v.y * g.inv_dt;
      }
      __syncthreads();
      continue;
    }
    // (5) conduction current J = (s dt_int) E, nodewise (a6, R17)
    {
      const uint8_t* sid = g.sig_id + (size_t)z * nx * ny;
      for (int t = tid; t < nline; t += bd) {
        const int p = t / ny, y = t - p * ny;
        float2 v = e[p * nyp + y];
        v.x *= g.sdt[sid[(2 * p) * ny + y]];
        v.y *= g.sdt[sid[(2 * p + 1) * ny + y]];
        e[p * nyp + y] = v;
      }
    }
    __syncthreads();
    // (6) forward along y
    float2* jf = wt::fft_lines<float2>(e, f, ny, hx, nyp, 1, g.twy, false);
    float2* jo = (jf == e) ? f : e;
    // (7) unpack the two real rows' half spectra
    for (int t = tid; t < hx * y2; t += bd) {
      const int p = t / y2, k = t - p * y2;
      const float2 zk = jf[p * nyp + k];
      const float2 zm = jf[p * nyp + (k == 0 ? 0 : ny - k)];
      jo[(2 * p) * y2 + k] = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
      jo[(2 * p + 1) * y2 + k] = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
    }
    __syncthreads();
    // (8) forward along x
    float2* jt = wt::fft_lines<float2>(jo, jf, nx, y2, 1, y2, g.twx, false);
    // (9) D~ = i kx J~x + i ky J~y ; J~z goes out as it is
    for (int t = tid; t < nspec; t += bd) {
      const int kx = t / y2, ky = t - kx * y2;
      const float2 j = jt[t];
      if (comp == 0) {
        const float kap = (float)g.kxd[kx];
        dacc[t] = make_float2(-kap * j.y, kap * j.x);
      } else if (comp == 1) {
        const float kap = (float)g.kyd[ky];
        float2 d = dacc[t];
        d.x -= kap * j.y; d.y += kap * j.x;
        dacc[t] = d;
      } else {
        const size_t gi = ((size_t)kx * nz + z) * y2 + ky;
        g.m1[gi] = j;
        g.m0[gi] = dacc[t];
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// k_transpose: staging [slot][comp][z][x][y] -> H[((x*ny+y)*nz+z)*nt + t][comp] for t0 <= t < t0+cnt.
// grid (nz*nx, n_geoms), block 256; dynamic smem cnt*3*ny floats.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_transpose(GridDev gd, const GeomDev* __restrict__ geoms, int t0, int cnt) {
  const GeomDev& g = geoms[blockIdx.y];
  const int nx = gd.nx, ny = gd.ny, nz = gd.nz, nt = gd.nt;
  const int z = blockIdx.x / nx, x = blockIdx.x - z * nx;
  extern __shared__ float tile[];   // [cnt*3][ny]
  const int rows = cnt * 3;
  for (int t = threadIdx.x; t < rows * ny; t += blockDim.x) {
    const int j = t / ny, y = t - j * ny;          // j = slot*3 + comp
    tile[t] = g.stage[(((size_t)j * nz + z) * nx + x) * ny + y];
  }
  __syncthreads();
  for (int t = threadIdx.x; t < rows * ny; t += blockDim.x) {
    const int y = t / rows, j = t - y * rows;
    g.H[((((size_t)x * ny + y) * nz + z) * nt + t0) * 3 + j] = tile[j * ny + y];
  }
}

__global__ void k_zero(double2* p, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = make_double2(0.0, 0.0);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

int pick_ty(int y2) {
  const int cand[6] = {8, 6, 4, 3, 2, 1};
  for (int c : cand)
    if (y2 % c == 0) return c;
  return 1;
}

// Offsets of one geometry's region inside the workspace (static tables, then state).
struct Layout {
  size_t sig_id, sdt, gt, gzt, ainv, pad_x, pad_y, pad_layer, pad_pot, layer_off, layer_idx;
  size_t kxd, kyd, kzd, twx, twy, twz, twxd, twyd, twzd;
  size_t rhat, rhat_prev, m0, m1, e0, e1, part, part_e, rhs, q, qh, stage;
  size_t total;
};

Layout make_layout(const wt_geometry* g) {
  Layout o;
  const size_t nx = g->nx, ny = g->ny, nz = g->nz, y2 = ny / 2;
  const size_t N = nx * ny * nz, half = nx * nz * y2;
  const size_t B = g->pad_pot.size(), L = g->layers.size();
  const size_t tiles = nx * (y2 / pick_ty((int)y2));
  size_t p = 0;
  auto take = [&](size_t bytes) { size_t at = p; p = align_up(p + bytes); return at; };
  o.sig_id = take(N); o.sdt = take(256 * 4); o.gt = take(half * 4); o.gzt = take(half * 4);
  o.ainv = take(B * B * 8); o.pad_x = take(B * 4); o.pad_y = take(B * 4); o.pad_layer = take(B * 4);
  o.pad_pot = take(B * 8); o.layer_off = take((L + 1) * 4); o.layer_idx = take(B * 4);
  o.kxd = take(nx * 8); o.kyd = take(y2 * 8); o.kzd = take(nz * 8);
  o.twx = take(nx * 8); o.twy = take(ny * 8); o.twz = take(nz * 8);
  o.twxd = take(nx * 16); o.twyd = take(ny * 16); o.twzd = take(nz * 16);
  o.rhat = take(half * 16); o.rhat_prev = take(half * 16);
  o.m0 = take(half * 8); o.m1 = take(half * 8); o.e0 = take(half * 8); o.e1 = take(half * 8);
  o.part = take(tiles * B * 8); o.part_e = take(tiles * B * 8);
  o.rhs = take(B * 8); o.q = take(B * 8); o.qh = take(L * nx * y2 * 8);
  o.stage = take((size_t)kStageSlots * 3 * N * 4);
  o.total = p;
  return o;
}

size_t spectral_smem(const wt_geometry* g) {
  const int y2 = g->ny / 2, ty = pick_ty(y2);
  const size_t L = g->layers.size();
  return (size_t)3 * g->nz * ty * 8 + (L * ty * 32 + L * ty) * 16;
}
size_t plane_smem(const wt_geometry* g) { return (size_t)3 * (g->nx / 2) * (g->ny + 1) * 8; }

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

}  // namespace

// bytes wt_solve_H needs for this geometry (its region + one descriptor slot)
size_t wt_solve_workspace_bytes(const wt_geometry* g) { return make_layout(g).total + align_up(sizeof(GeomDev)); }

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
  const size_t need = regions + align_up((size_t)n_geoms * sizeof(GeomDev));
  const size_t hbytes = (size_t)g0->nx * g0->ny * g0->nz * g0->nt * 12;
  if (H_bytes_each < hbytes) { wt_set_error("wt_solve_H: H_bytes_each too small"); return WT_EINVAL; }
  if (((uintptr_t)workspace_dev) % 256 != 0) { wt_set_error("wt_solve_H: workspace not 256-byte aligned"); return WT_EINVAL; }
  if (workspace_bytes < need) { wt_set_error("wt_solve_H: workspace too small, need " + std::to_string(need)); return WT_ENOMEM; }
  size_t sm_spec = 0;
  const size_t sm_plane = plane_smem(g0);
  for (int i = 0; i < n_geoms; ++i) sm_spec = std::max(sm_spec, spectral_smem(geoms[i]));
  if (sm_spec > 227 * 1024 || sm_plane > 227 * 1024) {
    wt_set_error("wt_solve_H: grid too large for the shared-memory tiles (nx*ny <= 128*128)"); return WT_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nx = g0->nx, ny = g0->ny, nz = g0->nz, y2 = ny / 2, nt = g0->nt;
  const int TY = pick_ty(y2);
  GridDev gd;
  gd.nx = nx; gd.ny = ny; gd.nz = nz; gd.y2 = y2; gd.nt = nt; gd.ty = TY; gd.n_tiles = nx * (y2 / TY);
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

  // ---- upload static tables, build the device descriptors ------------------------------------
  std::vector<GeomDev> hd(n_geoms);
  char* base = (char*)workspace_dev;
  size_t off = 0;
  int maxB = 0, maxL = 0;
  for (int i = 0; i < n_geoms; ++i) {
    const wt_geometry* g = geoms[i];
    const Layout lo = make_layout(g);
    char* b = base + off;
    const int B = (int)g->pad_pot.size(), L = (int)g->layers.size();
    maxB = std::max(maxB, B); maxL = std::max(maxL, L);
    std::vector<int> px(B), py(B), loff(L + 1, 0), lidx(B);
    for (int k = 0; k < B; ++k) { px[k] = g->pad_nodes[3 * k]; py[k] = g->pad_nodes[3 * k + 1]; }
    for (int k = 0; k < B; ++k) loff[g->pad_layer[k] + 1]++;
    for (int l = 0; l < L; ++l) loff[l + 1] += loff[l];
    {
      std::vector<int> cur(loff.begin(), loff.end() - 1);
      for (int k = 0; k < B; ++k) lidx[cur[g->pad_layer[k]]++] = k;
    }
    CK(upload(b, lo.sig_id, g->sig_id, st)); CK(upload(b, lo.sdt, g->sdt, st));
    CK(upload(b, lo.gt, g->gt, st)); CK(upload(b, lo.gzt, g->gzt, st));
    CK(upload(b, lo.ainv, g->ainv, st));
    CK(upload(b, lo.pad_x, px, st)); CK(upload(b, lo.pad_y, py, st));
    CK(upload(b, lo.pad_layer, g->pad_layer, st)); CK(upload(b, lo.pad_pot, g->pad_pot, st));
    CK(upload(b, lo.layer_off, loff, st)); CK(upload(b, lo.layer_idx, lidx, st));
    CK(upload(b, lo.kxd, g->kx, st)); CK(upload(b, lo.kyd, g->ky, st)); CK(upload(b, lo.kzd, g->kz, st));
    CK(upload(b, lo.twx, twx, st)); CK(upload(b, lo.twy, twy, st)); CK(upload(b, lo.twz, twz, st));
    CK(upload(b, lo.twxd, twxd, st)); CK(upload(b, lo.twyd, twyd, st)); CK(upload(b, lo.twzd, twzd, st));
    GeomDev& d = hd[i];
    d.sig_id = (const uint8_t*)(b + lo.sig_id); d.sdt = (const float*)(b + lo.sdt);
    d.gt = (const float*)(b + lo.gt); d.gzt = (const float*)(b + lo.gzt);
    d.ainv = (const double*)(b + lo.ainv);
    d.pad_x = (const int*)(b + lo.pad_x); d.pad_y = (const int*)(b + lo.pad_y);
    d.pad_layer = (const int*)(b + lo.pad_layer); d.pad_pot = (const double*)(b + lo.pad_pot);
    d.layer_off = (const int*)(b + lo.layer_off); d.layer_idx = (const int*)(b + lo.layer_idx);
    d.kxd = (const double*)(b + lo.kxd); d.kyd = (const double*)(b + lo.kyd); d.kzd = (const double*)(b + lo.kzd);
    d.twx = (const float2*)(b + lo.twx); d.twy = (const float2*)(b + lo.twy); d.twz = (const float2*)(b + lo.twz);
    d.twxd = (const double2*)(b + lo.twxd); d.twyd = (const double2*)(b + lo.twyd); d.twzd = (const double2*)(b + lo.twzd);
    d.rhat = (double2*)(b + lo.rhat); d.rhat_prev = (double2*)(b + lo.rhat_prev);
    d.m0 = (float2*)(b + lo.m0); d.m1 = (float2*)(b + lo.m1); d.e0 = (float2*)(b + lo.e0); d.e1 = (float2*)(b + lo.e1);
    d.part = (double*)(b + lo.part); d.part_e = (double*)(b + lo.part_e);
    d.rhs = (double*)(b + lo.rhs); d.q = (double*)(b + lo.q); d.qh = (float2*)(b + lo.qh);
    d.stage = (float*)(b + lo.stage);
    d.H = H_dev[i];
    for (int l = 0; l < kMaxLayers; ++l) d.layers[l] = (l < L) ? g->layers[l] : 0;
    d.B = B; d.L = L; d.n_sub = g->n_sub; d.inv_dt = (float)(1.0 / g->dt);
    off += lo.total;
  }
  GeomDev* dgeoms = (GeomDev*)(base + off);
  CK(cudaMemcpyAsync(dgeoms, hd.data(), (size_t)n_geoms * sizeof(GeomDev), cudaMemcpyHostToDevice, st));

  // ---- launch configuration -------------------------------------------------------------------
  CK(cudaFuncSetAttribute(k_spectral<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_spec));
  CK(cudaFuncSetAttribute(k_spectral<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_spec));
  CK(cudaFuncSetAttribute(k_spectral<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_spec));
  CK(cudaFuncSetAttribute(k_plane<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_plane));
  CK(cudaFuncSetAttribute(k_plane<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_plane));
  const dim3 g_spec(gd.n_tiles, n_geoms), b_spec(32 * TY);
  const dim3 g_plane(nz, n_geoms);
  const dim3 g_warpB((maxB * 32 + 255) / 256, n_geoms);
  const dim3 g_inj((nx * y2 + 255) / 256, maxL, n_geoms);
  const dim3 g_tr(nz * nx, n_geoms);
  const size_t half = (size_t)nx * nz * y2;

  auto boundary = [&](int s, int emit, double flag) {
    if (maxB == 0) return;
    g_wt_launches += 3;
    k_rhs<<<g_warpB, 256, 0, st>>>(gd, dgeoms, s, emit, flag);
    k_matvec<<<g_warpB, 256, 0, st>>>(dgeoms, s);
    k_inject<<<g_inj, 256, 0, st>>>(gd, dgeoms, s);
  };
  auto emit_step = [&](int n) {
    // H[n] from the increment of the charge since the previous output step (the prompt response
    // H[0] from the pads alone: r = 0, pads at v_w)
    g_wt_launches += 2;
    if (n == 0) k_spectral<false, false><<<g_spec, b_spec, sm_spec, st>>>(gd, dgeoms, 0, 1);
    else        k_spectral<false, true><<<g_spec, b_spec, sm_spec, st>>>(gd, dgeoms, 0, 1);
    boundary(0, 1, n == 0 ? 1.0 : 0.0);
    k_plane<true><<<g_plane, 256, sm_plane, st>>>(gd, dgeoms, 0, n % kStageSlots);
    if ((n + 1) % kStageSlots == 0 || n == nt - 1) {
      const int cnt = n % kStageSlots + 1, t0 = n - cnt + 1;
      ++g_wt_launches;
      k_transpose<<<g_tr, 256, (size_t)cnt * 3 * ny * sizeof(float), st>>>(gd, dgeoms, t0, cnt);
    }
  };

  g_wt_launches += 2 * n_geoms + 1;
  for (int i = 0; i < n_geoms; ++i) {
    k_zero<<<(unsigned)((half + 255) / 256), 256, 0, st>>>(hd[i].rhat, half);
    k_zero<<<(unsigned)((half + 255) / 256), 256, 0, st>>>(hd[i].rhat_prev, half);
    if (maxL > 0) CK(cudaMemsetAsync(hd[i].qh, 0, (size_t)hd[i].L * nx * y2 * sizeof(float2), st));
  }
  emit_step(0);
  k_spectral<false, false><<<g_spec, b_spec, sm_spec, st>>>(gd, dgeoms, 0, 0);
  for (int n = 1; n < nt; ++n) {
    for (int s = 0; s < max_sub; ++s) {
      boundary(s, 0, 1.0);
      g_wt_launches += 2;
      k_plane<false><<<g_plane, 256, sm_plane, st>>>(gd, dgeoms, s, 0);
      k_spectral<true, false><<<g_spec, b_spec, sm_spec, st>>>(gd, dgeoms, s, 0);
    }
    emit_step(n);
  }
  CK(cudaGetLastError());
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
