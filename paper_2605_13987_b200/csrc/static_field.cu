// wt_solve_static: SURVEY 8(f) row 1 -- the electrostatic (Laplace) field of the sensor, PAPER.md:64 ("An iterative
// pseudo-spectral method ... is used to solve the Laplace equation in the diamond sensor"), :95 (V <-> rho through the 3-D FFT
// and a kernel that multiplies or divides by |k|^2), Fig. 2 (:107).  Reading R37 of DESIGN.md: every node of column j is held
// at potential v_j, there is no charge elsewhere, the box is periodic and neutral:
//     V(x) = c + sum_{s in S} q_s G(x - x_s),   V(x_s) = v_s on S,   sum_s q_s = 0,
// G the fundamental solution of the same spectral Laplacian (Nyquist modes removed, R11).  The iteration is conjugate
// gradients on the restricted operator  P G P^T  in the neutral subspace (projector Pi = I - 11^T/|S|), optionally
// preconditioned by the restricted Laplacian  P |k|^2 P^T  (the "rho from V" direction of Fig. 2): each step is one
// V <-> rho round trip -- forward 3-D DFT, times 1/|k|^2 or |k|^2, inverse 3-D DFT, restriction to the electrodes.
//
// Execution: ONE cooperative launch for the whole solve.  CTAs own xy-planes (real 2-D transforms, two x-rows packed into a
// complex line) and z-line tiles (kx, TY ky); the phases of a round trip are separated by grid barriers, the CG scalars are
// formed by every CTA from per-plane partial sums in a fixed order (bitwise identical on every CTA, so all CTAs take the
// same branch and the result is run-to-run deterministic).  Transforms are fp32 (fft.cuh), the CG vectors and all sums fp64.
// The working set (41 B per node) stays in L2 for the BASELINE grids.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

#include "fft.cuh"
#include "geometry.h"

namespace wt {
namespace {

constexpr int kStThreads = 256;
constexpr int kMaxIds = 256;                       // column ids are uint8: 0 = diamond, j + 1 = column j
constexpr long long kStSpinLimit = 4000000000LL;   // cycles (about two seconds): a lost CTA aborts the solve instead of hanging it

struct StaticCtl {
  unsigned long long bar;
  int abort;
  int pad;
};

struct StaticArgs {
  int nx, ny, nz, y2, ty, max_iter, precond;
  double n_s;                  // |S|, number of electrode nodes
  double inv_n, tol2;
  const uint8_t* mask;         // [z][x][y]
  const double* pot;           // [256] potential of id
  const double *kx, *ky, *kz;  // wavenumbers (0 at the removed Nyquist index); ky has y2 entries
  double *q, *r, *p, *w;       // [z][x][y]: charges, residual, search direction, operator output
  float2 *m0, *m1;             // [kx][z][ky] mixed-space fields
  double* part;                // [nz][2] per-plane partial sums
  StaticCtl* ctl;
  float* V;                    // [nx][ny][nz] or NULL
  float* E;                    // [nx*ny*nz][3] or NULL
  double* info;                // [4]: iterations (-1: aborted), relative residual, c, sum of q'
};

__device__ __forceinline__ unsigned long long st_ld_acquire(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

struct Smem {
  float2 *w1, *w2, *w3;        // plane: two buffers of hx*(ny+1); z tile: three of nz*ty (overlaid)
  float2 *twx, *twy, *twz;
  double* red;                 // [2 * kStThreads/32 + 2]
  double* kz;                  // [nz] z wavenumbers (z tiles read one per mode)
  int* flag;
};

// ---- 2-D real transforms of one plane (structure of k_plane, solve_generic.cuh) -------------------------------
// forward: src(x, y) real -> half spectrum M[kx][z][ky], ky < y2 (the y Nyquist column is dropped: R11)
template <typename Src>
__device__ __forceinline__ void plane_forward(const StaticArgs& a, const Smem& s, int z, Src src, float2* __restrict__ M) {
  const int nx = a.nx, ny = a.ny, nz = a.nz, y2 = a.y2, hx = nx / 2, nyp = ny + 1;
  const int tid = threadIdx.x, bd = blockDim.x;
  for (int t = tid; t < hx * ny; t += bd) {
    const int p = t / ny, y = t - p * ny;
    s.w1[p * nyp + y] = make_float2(src(2 * p, y), src(2 * p + 1, y));
  }
  __syncthreads();
  float2* jf = fft_lines<float2>(s.w1, s.w2, ny, hx, nyp, 1, s.twy, false);
  float2* jo = (jf == s.w1) ? s.w2 : s.w1;
  for (int t = tid; t < hx * y2; t += bd) {
    const int p = t / y2, k = t - p * y2;
    const float2 zk = jf[p * nyp + k];
    const float2 zm = jf[p * nyp + (k == 0 ? 0 : ny - k)];
    jo[(2 * p) * y2 + k] = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
    jo[(2 * p + 1) * y2 + k] = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
  }
  __syncthreads();
  float2* jt = fft_lines<float2>(jo, jf, nx, y2, 1, y2, s.twx, false);
  for (int t = tid; t < nx * y2; t += bd) {
    const int kx = t / y2, ky = t - kx * y2;
    M[((size_t)kx * nz + z) * y2 + ky] = jt[t];
  }
  __syncthreads();
}

// inverse: load(kx, ky) -> real plane; returns the buffer e with e[p*(ny+1) + y] = (f(2p, y), f(2p+1, y))
template <typename Load>
__device__ __forceinline__ float2* plane_inverse(const StaticArgs& a, const Smem& s, Load load) {
  const int nx = a.nx, ny = a.ny, y2 = a.y2, hx = nx / 2, nyp = ny + 1;
  const int tid = threadIdx.x, bd = blockDim.x;
  for (int t = tid; t < nx * y2; t += bd) {
    const int kx = t / y2, ky = t - kx * y2;
    s.w1[t] = load(kx, ky);
  }
  __syncthreads();
  float2* r = fft_lines<float2>(s.w1, s.w2, nx, y2, 1, y2, s.twx, true);
  float2* o = (r == s.w1) ? s.w2 : s.w1;
  for (int t = tid; t < hx * ny; t += bd) {
    const int p = t / ny, k = t - p * ny;
    float2 zv;
    if (k < y2) {
      const float2 u = r[(2 * p) * y2 + k], v = r[(2 * p + 1) * y2 + k];
      zv = make_float2(u.x - v.y, u.y + v.x);
    } else if (k == y2) {
      zv = make_float2(0.f, 0.f);
    } else {
      const float2 u = r[(2 * p) * y2 + (ny - k)], v = r[(2 * p + 1) * y2 + (ny - k)];
      zv = make_float2(u.x + v.y, v.x - u.y);
    }
    o[p * nyp + k] = zv;
  }
  __syncthreads();
  return fft_lines<float2>(o, r, ny, hx, nyp, 1, s.twy, true);
}

// ---- z-line tile: forward z, spectral multiplier, inverse z -------------------------------------------------
// MODE 0: times 1/|k|^2 (V from rho), 1: times |k|^2 (rho from V), 2: as 0 and also -i kz V^ -> m1 (final field)
template <int MODE>
__device__ __forceinline__ void z_tile(const StaticArgs& a, const Smem& s, int tile) {
  const int nx = a.nx, nz = a.nz, y2 = a.y2, TY = a.ty;
  const int tiles = y2 / TY;
  const int kx = tile / tiles, ky0 = (tile - kx * tiles) * TY;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int nelem = nz * TY;
  const size_t slab = (size_t)kx * nz * y2 + ky0;
  for (int t = tid; t < nelem; t += bd) {
    const int z = t / TY, ty = t - z * TY;
    s.w1[t] = __ldcg(a.m0 + slab + (size_t)z * y2 + ty);
  }
  __syncthreads();
  float2* f = fft_lines<float2>(s.w1, s.w2, nz, TY, 1, TY, s.twz, false);
  float2* o = (f == s.w1) ? s.w2 : s.w1;
  const double kxd = a.kx[kx];
  const bool ret_x = (kx != nx / 2);
  for (int t = tid; t < nelem; t += bd) {
    const int kz = t / TY, ty = t - kz * TY;
    const double kyd = a.ky[ky0 + ty], kzd = s.kz[kz];
    const bool ret = ret_x && (kz != nz / 2);
    const double k2 = kxd * kxd + kyd * kyd + kzd * kzd;
    double m;
    if (MODE == 1) m = ret ? a.inv_n * k2 : 0.0;
    else m = (ret && k2 > 0.0) ? a.inv_n / k2 : 0.0;
    const float2 v = f[t];
    const float2 u = make_float2((float)(m * (double)v.x), (float)(m * (double)v.y));
    f[t] = u;
    if (MODE == 2) {
      const float kzf = (float)kzd;
      s.w3[t] = make_float2(kzf * u.y, -kzf * u.x);     // -i kz V^
    }
  }
  __syncthreads();
  float2* v = fft_lines<float2>(f, o, nz, TY, 1, TY, s.twz, true);
  for (int t = tid; t < nelem; t += bd) {
    const int z = t / TY, ty = t - z * TY;
    a.m0[slab + (size_t)z * y2 + ty] = v[t];
  }
  if (MODE == 2) {
    float2* fr = (v == f) ? o : f;
    __syncthreads();
    float2* e = fft_lines<float2>(s.w3, fr, nz, TY, 1, TY, s.twz, true);
    for (int t = tid; t < nelem; t += bd) {
      const int z = t / TY, ty = t - z * TY;
      a.m1[slab + (size_t)z * y2 + ty] = e[t];
    }
  }
  __syncthreads();
}

// block sum of two doubles in a fixed order; the result is returned to every thread
__device__ __forceinline__ void block_sum2(double& x, double& y, double* red) {
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    x += __shfl_down_sync(0xffffffffu, x, o);
    y += __shfl_down_sync(0xffffffffu, y, o);
  }
  if (lane == 0) { red[2 * wid] = x; red[2 * wid + 1] = y; }
  __syncthreads();
  if (tid == 0) {
    double sx = 0.0, sy = 0.0;
    for (int i = 0; i < nw; ++i) { sx += red[2 * i]; sy += red[2 * i + 1]; }
    red[2 * nw] = sx; red[2 * nw + 1] = sy;
  }
  __syncthreads();
  x = red[2 * nw]; y = red[2 * nw + 1];
  __syncthreads();
}

// ------------------------------------------------------------------------------------------------
// k_static_cg: the whole Laplace solve.  grid = co-resident CTAs (cooperative launch), block 256.
// ------------------------------------------------------------------------------------------------
// NXY, NZC: the grids of BASELINE configs[1] / [3] (64 x 64 x 256), [2] (128 x 128 x 256) and [4] (96 x 96 x 384), 8 lines per z tile, with
// compile-time sizes, so that the index arithmetic of the Stockham passes and of the pack / unpack loops folds to constants
// (87 -> 72 us per iteration at configs[1]); NXY = 0: the sizes are run-time values
template <int NXY, int NZC>
__global__ void __launch_bounds__(kStThreads) k_static_cg(const __grid_constant__ StaticArgs a_in) {
  StaticArgs a = a_in;
  if constexpr (NXY != 0) { a.nx = NXY; a.ny = NXY; a.nz = NZC; a.y2 = NXY / 2; a.ty = 8; }
  extern __shared__ __align__(16) unsigned char smraw[];
  const int nx = a.nx, ny = a.ny, nz = a.nz, y2 = a.y2, hx = nx / 2, nyp = ny + 1;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int cta = blockIdx.x, n_cta = gridDim.x;
  const int n_tiles = nx * (y2 / a.ty);
  Smem s;
  {
    const size_t plane_buf = (size_t)hx * nyp, z_buf = (size_t)nz * a.ty;
    const size_t work = (2 * plane_buf > 3 * z_buf) ? 2 * plane_buf : 3 * z_buf;
    float2* base = reinterpret_cast<float2*>(smraw);
    s.w1 = base;
    // (plane phases use w1, w2 with stride plane_buf; z phases w1, w2, w3 with stride z_buf)
    s.w2 = base + plane_buf; s.w3 = nullptr;
    s.twx = base + work; s.twy = s.twx + nx; s.twz = s.twy + ny;
    s.red = reinterpret_cast<double*>(s.twz + nz);
    s.kz = s.red + 2 * (kStThreads / 32) + 2;
    s.flag = reinterpret_cast<int*>(s.kz + nz);
  }
  Smem sz = s;                                       // z-phase view of the same memory
  sz.w2 = s.w1 + (size_t)nz * a.ty; sz.w3 = sz.w2 + (size_t)nz * a.ty;
  for (int i = tid; i < nz; i += bd) s.kz[i] = a.kz[i];
  for (int i = tid; i < nx + ny + nz; i += bd) {     // twiddles e^{-2 pi i k/n}
    const int n = (i < nx) ? nx : (i < nx + ny ? ny : nz);
    const int k = (i < nx) ? i : (i < nx + ny ? i - nx : i - nx - ny);
    double sn, cs;
    sincospi(2.0 * (double)k / (double)n, &sn, &cs);
    s.twx[i] = make_float2((float)cs, (float)(-sn));
  }
  __syncthreads();

  unsigned long long bar_n = 0;
  auto grid_barrier = [&]() -> bool {
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      atomicAdd(&a.ctl->bar, 1ULL);
      ++bar_n;
      const unsigned long long target = bar_n * (unsigned long long)n_cta;
      const long long t0 = clock64();
      unsigned it = 0;
      int ok = 1;
      while (st_ld_acquire(&a.ctl->bar) < target) {
        if ((++it & 63u) == 0) {
          if (*reinterpret_cast<volatile int*>(&a.ctl->abort)) { ok = 0; break; }
          if (clock64() - t0 > kStSpinLimit) { atomicExch(&a.ctl->abort, 1); ok = 0; break; }
        }
      }
      *s.flag = ok;
    }
    __syncthreads();
    const bool ok = *s.flag != 0;
    __syncthreads();
    return ok;
  };
  // sum of the per-plane partials, fixed order: identical bits on every CTA
  auto reduce_parts = [&](double& x, double& y) {
    double sx = 0.0, sy = 0.0;
    for (int z = tid; z < nz; z += bd) { sx += __ldcg(a.part + 2 * z); sy += __ldcg(a.part + 2 * z + 1); }
    block_sum2(sx, sy, s.red);
    x = sx; y = sy;
  };
  // for each electrode node of plane z: fn(index in the [z][x][y] arrays, potential of the node)
  auto plane_nodes = [&](int z, auto fn) {
    const size_t base = (size_t)z * nx * ny;
    for (int t = tid; t < nx * ny; t += bd) {
      const uint8_t id = a.mask[base + t];
      if (id) fn(base + t, id);
    }
  };
  auto put_part = [&](int z, double x, double y) {
    block_sum2(x, y, s.red);
    if (tid == 0) { a.part[2 * z] = x; a.part[2 * z + 1] = y; }
  };

  // SRC 0: p <- (PRE ? w - mean_z : r) + beta p, transform p;  1: transform r;  2: transform q
  auto phase_forward = [&](int src_kind, bool pre, double mean_z, double beta) {
    for (int z = cta; z < nz; z += n_cta) {
      const size_t base = (size_t)z * nx * ny;
      if (src_kind == 0) {
        plane_nodes(z, [&](size_t i, uint8_t) {
          const double zz = pre ? (__ldcg(a.w + i) - mean_z) : __ldcg(a.r + i);
          a.p[i] = zz + beta * __ldcg(a.p + i);
        });
        __syncthreads();
      }
      const double* v = (src_kind == 0) ? a.p : (src_kind == 1 ? a.r : a.q);
      plane_forward(a, s, z, [&](int x, int y) -> float {
        const size_t i = base + (size_t)x * ny + y;
        return a.mask[i] ? (float)__ldcg(v + i) : 0.f;
      }, a.m0);
    }
  };
  auto phase_z = [&](int mode) {
    for (int t = cta; t < n_tiles; t += n_cta) {
      if (mode == 0) z_tile<0>(a, sz, t);
      else if (mode == 1) z_tile<1>(a, sz, t);
      else z_tile<2>(a, sz, t);
    }
  };
  // w <- restriction of the inverse transform; partial sums (sum dotv * w, sum w) per plane
  auto phase_inverse = [&](const double* dotv) {
    for (int z = cta; z < nz; z += n_cta) {
      const float2* e = plane_inverse(a, s, [&](int kx, int ky) { return __ldcg(a.m0 + ((size_t)kx * nz + z) * y2 + ky); });
      const size_t base = (size_t)z * nx * ny;
      double d = 0.0, sw = 0.0;
      for (int t = tid; t < nx * ny; t += bd) {
        if (!a.mask[base + t]) continue;
        const int x = t / ny, y = t - x * ny;
        const float2 v = e[(x >> 1) * nyp + y];
        const double val = (x & 1) ? (double)v.y : (double)v.x;
        a.w[base + t] = val;
        d += __ldcg(dotv + base + t) * val;
        sw += val;
      }
      put_part(z, d, sw);     // (its barriers also protect e before the next plane's loads)
    }
  };

  // ---- right-hand side b = Pi v, start q = 0, r = b, p = 0 ------------------------------------------------------
  for (int z = cta; z < nz; z += n_cta) {
    double sb = 0.0, zero = 0.0;
    plane_nodes(z, [&](size_t, uint8_t id) { sb += a.pot[id]; });
    put_part(z, sb, zero);
  }
  if (!grid_barrier()) return;
  double sum_b, dummy;
  reduce_parts(sum_b, dummy);
  const double mean_b = sum_b / a.n_s;
  for (int z = cta; z < nz; z += n_cta) {
    double rr = 0.0, zero = 0.0;
    plane_nodes(z, [&](size_t i, uint8_t id) {
      const double b = a.pot[id] - mean_b;
      a.r[i] = b; a.q[i] = 0.0; a.p[i] = 0.0;
      rr += b * b;
    });
    put_part(z, rr, zero);
  }
  if (!grid_barrier()) return;
  double bb;
  reduce_parts(bb, dummy);

  // ---- conjugate gradients on Pi (P G P^T) Pi q = b, preconditioner Pi (P |k|^2 P^T) Pi ---------------------------
  const bool pre = a.precond != 0;
  double rr = bb, rz = bb, beta = 0.0, mean_z = 0.0, sum_r = 0.0;
  int it = 0;
  bool live = bb > 0.0 && a.max_iter > 0;
  if (live && pre) {
    phase_forward(1, false, 0.0, 0.0);
    if (!grid_barrier()) return;
    phase_z(1);
    if (!grid_barrier()) return;
    phase_inverse(a.r);
    if (!grid_barrier()) return;
    double sz_;
    reduce_parts(rz, sz_);
    mean_z = sz_ / a.n_s;
  }
  while (live) {
    phase_forward(0, pre, mean_z, beta);
    if (!grid_barrier()) return;
    phase_z(0);
    if (!grid_barrier()) return;
    phase_inverse(a.p);
    if (!grid_barrier()) return;
    double pap, sap;
    reduce_parts(pap, sap);
    if (!(pap > 0.0)) break;                         // (breakdown: the direction lies in the null space)
    const double alpha = rz / pap, mean_ap = sap / a.n_s;
    for (int z = cta; z < nz; z += n_cta) {
      double s2 = 0.0, s1 = 0.0;
      plane_nodes(z, [&](size_t i, uint8_t) {
        const double pi = __ldcg(a.p + i);
        a.q[i] = __ldcg(a.q + i) + alpha * pi;
        const double ri = __ldcg(a.r + i) - alpha * (__ldcg(a.w + i) - mean_ap);
        a.r[i] = ri;
        s2 += ri * ri; s1 += ri;
      });
      put_part(z, s2, s1);
      if (pre) {               // the preconditioner's round trip starts on the new residual of this plane at once (no barrier)
        const size_t base = (size_t)z * nx * ny;
        plane_forward(a, s, z, [&](int x, int y) -> float {
          const size_t i = base + (size_t)x * ny + y;
          return a.mask[i] ? (float)__ldcg(a.r + i) : 0.f;
        }, a.m0);
      }
    }
    if (!grid_barrier()) return;
    reduce_parts(rr, sum_r);
    ++it;
    if (rr <= a.tol2 * bb || it >= a.max_iter) break;
    double rzn = rr;
    if (pre) {
      phase_z(1);
      if (!grid_barrier()) return;
      phase_inverse(a.r);
      if (!grid_barrier()) return;
      double sz_;
      reduce_parts(rzn, sz_);
      mean_z = sz_ / a.n_s;
      rzn -= mean_z * sum_r;                         // r . (z - mean_z)
      if (!(rzn > 0.0)) break;
    }
    beta = rzn / rz;
    rz = rzn;
  }

  // ---- the field of the charges: V = c + G q, E = -grad_s V -------------------------------------------------------
  phase_forward(2, false, 0.0, 0.0);
  if (!grid_barrier()) return;
  phase_z(2);
  if (!grid_barrier()) return;
  // c = mean over the electrodes of (v - G q); sum of the charges
  for (int z = cta; z < nz; z += n_cta) {
    const float2* e = plane_inverse(a, s, [&](int kx, int ky) { return __ldcg(a.m0 + ((size_t)kx * nz + z) * y2 + ky); });
    double sd = 0.0, sq = 0.0;
    plane_nodes(z, [&](size_t i, uint8_t id) {
      const int t = (int)(i - (size_t)z * nx * ny), x = t / ny, y = t - x * ny;
      const float2 v = e[(x >> 1) * nyp + y];
      sd += a.pot[id] - ((x & 1) ? (double)v.y : (double)v.x);
      sq += __ldcg(a.q + i);
    });
    put_part(z, sd, sq);
  }
  if (!grid_barrier()) return;
  double sum_d, sum_q;
  reduce_parts(sum_d, sum_q);
  const float c = (float)(sum_d / a.n_s);
  for (int z = cta; z < nz; z += n_cta) {
    for (int comp = (a.V ? 0 : 1); comp < (a.E ? 4 : 1); ++comp) {
      const float2* e = plane_inverse(a, s, [&](int kx, int ky) {
        const size_t gi = ((size_t)kx * nz + z) * y2 + ky;
        if (comp == 3) return __ldcg(a.m1 + gi);
        const float2 v = __ldcg(a.m0 + gi);
        if (comp == 0) return v;
        const float kap = (comp == 1) ? (float)a.kx[kx] : (float)a.ky[ky];
        return make_float2(kap * v.y, -kap * v.x);                 // -i kappa V~
      });
      for (int t = tid; t < nx * ny; t += bd) {
        const int x = t / ny, y = t - x * ny;
        const float2 v = e[(x >> 1) * nyp + y];
        const float val = (x & 1) ? v.y : v.x;
        const size_t node = ((size_t)x * ny + y) * nz + z;
        if (comp == 0) a.V[node] = val + c;
        else a.E[node * 3 + (comp - 1)] = val;
      }
      __syncthreads();
    }
  }
  if (cta == 0 && tid == 0) {
    a.info[0] = (double)it;
    a.info[1] = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    a.info[2] = sum_d / a.n_s;
    a.info[3] = sum_q;
  }
}

__global__ void k_static_finish(StaticCtl* ctl, double* info) {
  if (ctl->abort) info[0] = -1.0;
}

struct StLayout {
  size_t mask, tab, q, r, p, w, m0, m1, part, ctl, total;
};

StLayout st_layout(const wt_geometry* g) {
  StLayout o;
  const size_t nx = g->nx, ny = g->ny, nz = g->nz, N = nx * ny * nz, half = nx * nz * (ny / 2);
  size_t p = 0;
  auto take = [&](size_t bytes) { size_t at = p; p = (p + bytes + 255) / 256 * 256; return at; };
  o.mask = take(N);
  o.tab = take((nx + ny / 2 + nz + kMaxIds) * 8);
  o.q = take(N * 8); o.r = take(N * 8); o.p = take(N * 8); o.w = take(N * 8);
  o.m0 = take(half * 8); o.m1 = take(half * 8);
  o.part = take(nz * 16);
  o.ctl = take(256);
  o.total = p;
  return o;
}

int pick_ty(int y2, int nz) {
  const int cap = std::max(1, std::min(8, 4096 / nz));
  int ty = 1;
  for (int t = 1; t <= cap; ++t)
    if (y2 % t == 0) ty = t;
  return ty;
}

size_t st_smem(const wt_geometry* g, int ty) {
  const size_t plane = (size_t)2 * (g->nx / 2) * (g->ny + 1), zt = (size_t)3 * g->nz * ty;
  return (std::max(plane, zt) + g->nx + g->ny + g->nz) * 8 + (2 * (kStThreads / 32) + 2) * 8 + (size_t)g->nz * 8 + 16;
}

int st_fail(const std::string& msg, int code) { wt_set_error("wt_solve_static: " + msg); return code; }

}  // namespace
}  // namespace wt

using namespace wt;

extern "C" int wt_static_workspace_bytes(const wt_geometry* g, size_t* bytes) {
  if (!wt_valid(g) || !bytes) { wt_set_error("wt_static_workspace_bytes: bad argument"); return WT_EINVAL; }
  *bytes = st_layout(g).total;
  return WT_OK;
}

extern "C" int wt_solve_static(const wt_geometry* g, const double* column_potentials, int n_potentials, int precondition, int max_iter,
                               double tol, float* V_dev, float* E_dev, double* info_dev, void* workspace_dev, size_t workspace_bytes,
                               void* cuda_stream) {
  if (!wt_valid(g) || !column_potentials || !info_dev || !workspace_dev || !cuda_stream || (!V_dev && !E_dev))
    return st_fail("bad argument, both outputs NULL, or NULL (default) stream", WT_EINVAL);
  if (n_potentials != g->n_columns) return st_fail("one potential per column of the descriptor is needed", WT_EINVAL);
  if (max_iter < 0 || !(tol >= 0.0)) return st_fail("max_iter < 0 or tol < 0", WT_EINVAL);
  if (((uintptr_t)workspace_dev) % 256 != 0) return st_fail("workspace not 256-byte aligned", WT_EINVAL);
  const StLayout lo = st_layout(g);
  if (workspace_bytes < lo.total) return st_fail("workspace too small, need " + std::to_string(lo.total), WT_ENOMEM);
  if (g->n_conducting < 1) return st_fail("no electrode node", WT_EGEOM);
  const int nx = g->nx, ny = g->ny, nz = g->nz, y2 = ny / 2;
  const int ty = pick_ty(y2, nz);
  const size_t smem = st_smem(g, ty);
  int dev = 0, n_sm = 0, max_smem = 0, coop = 0;
#define CKS(call)                                                                                  \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return st_fail(std::string(cudaGetErrorString(e_)) + " at " #call, WT_ECUDA); \
  } while (0)
  CKS(cudaGetDevice(&dev));
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  if (!coop) return st_fail("device without cooperative launch", WT_ECUDA);
  if (smem > (size_t)max_smem) return st_fail("an xy-plane of this grid does not fit in shared memory", WT_EINVAL);
  const void* fn = (const void*)k_static_cg<0, 0>;
  if (nx == ny && ty == 8) {
    if (nx == 64 && nz == 256) fn = (const void*)k_static_cg<64, 256>;
    else if (nx == 128 && nz == 256) fn = (const void*)k_static_cg<128, 256>;
    else if (nx == 96 && nz == 384) fn = (const void*)k_static_cg<96, 384>;
  }
  CKS(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  CKS(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, kStThreads, smem));
  if (per_sm < 1) return st_fail("kernel does not fit an SM", WT_ECUDA);
  const int n_tiles = nx * (y2 / ty);
  const int grid = std::min(n_sm * per_sm, std::max(nz, n_tiles));

  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* b = (char*)workspace_dev;
  // tables: wavenumbers and the potential of each column id, one small copy; the column map, one copy
  std::vector<double> tab((size_t)nx + y2 + nz + kMaxIds, 0.0);
  std::memcpy(tab.data(), g->kx.data(), (size_t)nx * 8);
  std::memcpy(tab.data() + nx, g->ky.data(), (size_t)y2 * 8);
  std::memcpy(tab.data() + nx + y2, g->kz.data(), (size_t)nz * 8);
  for (int j = 0; j < g->n_columns; ++j) tab[(size_t)nx + y2 + nz + 1 + j] = column_potentials[j];
  CKS(cudaMemcpyAsync(b + lo.tab, tab.data(), tab.size() * 8, cudaMemcpyHostToDevice, st));
  CKS(cudaMemcpyAsync(b + lo.mask, g->sig_id.data(), g->sig_id.size(), cudaMemcpyHostToDevice, st));
  CKS(cudaMemsetAsync(b + lo.ctl, 0, 256, st));
  CKS(cudaMemsetAsync(info_dev, 0, 4 * sizeof(double), st));

  StaticArgs a = {};
  a.nx = nx; a.ny = ny; a.nz = nz; a.y2 = y2; a.ty = ty; a.max_iter = max_iter; a.precond = precondition ? 1 : 0;
  a.n_s = (double)g->n_conducting;
  a.inv_n = 1.0 / ((double)nx * ny * nz); a.tol2 = tol * tol;
  a.mask = (const uint8_t*)(b + lo.mask);
  const double* t0 = (const double*)(b + lo.tab);
  a.kx = t0; a.ky = t0 + nx; a.kz = t0 + nx + y2; a.pot = t0 + nx + y2 + nz;
  a.q = (double*)(b + lo.q); a.r = (double*)(b + lo.r); a.p = (double*)(b + lo.p); a.w = (double*)(b + lo.w);
  a.m0 = (float2*)(b + lo.m0); a.m1 = (float2*)(b + lo.m1);
  a.part = (double*)(b + lo.part); a.ctl = (StaticCtl*)(b + lo.ctl);
  a.V = V_dev; a.E = E_dev; a.info = info_dev;
  void* kargs[] = {(void*)&a};
  CKS(cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(kStThreads), kargs, smem, st));
  k_static_finish<<<1, 1, 0, st>>>(a.ctl, info_dev);
  CKS(cudaGetLastError());
  g_wt_launches += 2;
  wt_set_error("");
  return WT_OK;
#undef CKS
}
