// Boundary adjust of wt_solve_H (steps a3, a4): the point charges on the pad nodes are "adjusted,
// in magnitude, to enforce the boundary conditions" (R8-R10 exact collocation).
//
//   k_padpot   V_rho at every pad node from the fp64 mixed-space planes pl[l][kx][ky] = V~_rho(kx, z_l, ky)
//              (written by the z-line kernel), evaluated separably: first along kx for each distinct pad
//              x of the layer, then along ky per pad;  rhs = flag * V_pad - V_rho|_B
//   k_matvec   Q' = Ainv rhs (fp64, one warp per row)
//   k_inject   Q^_l(kx,ky) = (1/N) sum_{b in layer l} Q'_b e^{-i(kx x_b + ky y_b)}, separably again
//              (along y per pad column, then along x); the plane kernel multiplies it with the
//              translated fundamental solution g~(kx, z - z_l, ky)  (the paper's V_ext, O(N) instead of O(|B| N))
#pragma once
#include "solve_common.cuh"

namespace wt {

constexpr int kPadChunks = 8;   // kx range split of k_padpot's first phase
constexpr int kInjKx = 8;       // kx values per CTA of k_inject

// grid (G_max, n_geoms), block 256, dynamic smem (kPadChunks + 1) * y2 * sizeof(double2)
__global__ void __launch_bounds__(256) k_padpot(GridDev gd, const GeomDev* __restrict__ geoms, int substep, int emit, double flag) {
  const GeomDev& g = geoms[blockIdx.y];
  if (substep >= g.n_sub || (int)blockIdx.x >= g.G) return;
  const int grp = blockIdx.x, l = g.grp_layer[grp], x = g.grp_x[grp];
  const int nx = gd.nx, ny = gd.ny, y2 = gd.y2, tid = threadIdx.x;
  extern __shared__ __align__(16) unsigned char smraw[];
  double2* part = reinterpret_cast<double2*>(smraw);   // [kPadChunks][y2]
  double2* tl = part + kPadChunks * y2;                // [y2]
  const double2* pl = (emit ? g.pl_e : g.pl) + (size_t)l * nx * y2;
  const int per = (nx + kPadChunks - 1) / kPadChunks;
  for (int i = tid; i < y2 * kPadChunks; i += 256) {
    const int ky = i % y2, ch = i / y2;
    const int k0 = ch * per, k1 = min(nx, k0 + per);
    double2 s = make_double2(0.0, 0.0);
    for (int kx = k0; kx < k1; ++kx) {
      double2 w = g.twxd[(kx * x) % nx];
      w.y = -w.y;                                       // e^{+i kx x}
      const double2 p = dmul(pl[(size_t)kx * y2 + ky], w);
      s.x += p.x; s.y += p.y;
    }
    part[ch * y2 + ky] = s;
  }
  __syncthreads();
  for (int ky = tid; ky < y2; ky += 256) {
    double2 s = make_double2(0.0, 0.0);
#pragma unroll
    for (int ch = 0; ch < kPadChunks; ++ch) { const double2 p = part[ch * y2 + ky]; s.x += p.x; s.y += p.y; }
    const double wgt = (ky == 0) ? 1.0 : 2.0;           // Hermitian half spectrum along y
    tl[ky] = make_double2(wgt * s.x, wgt * s.y);
  }
  __syncthreads();
  const int warp = tid >> 5, lane = tid & 31;
  for (int i = g.grp_off[grp] + warp; i < g.grp_off[grp + 1]; i += 8) {
    const int b = g.grp_pad[i], y = g.pad_y[b];
    double s = 0.0;
    for (int ky = lane; ky < y2; ky += 32) {
      const double2 w = g.twyd[(ky * y) % ny];           // Re(T e^{+i ky y}) = T.x w.x + T.y w.y with w = e^{-i ky y}
      const double2 t = tl[ky];
      s += t.x * w.x + t.y * w.y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) g.rhs[b] = flag * g.pad_pot[b] - s;
  }
}

// one warp per row of Ainv; grid (ceil(B_max/8), n_geoms), block 256
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

// grid (ceil(nx/kInjKx), L_max, n_geoms), block 256, dynamic smem (max groups per layer) * y2 * sizeof(double2)
__global__ void __launch_bounds__(256) k_inject(GridDev gd, const GeomDev* __restrict__ geoms, int substep) {
  const GeomDev& g = geoms[blockIdx.z];
  if (substep >= g.n_sub) return;
  const int l = blockIdx.y;
  if (l >= g.L) return;
  const int nx = gd.nx, ny = gd.ny, y2 = gd.y2, tid = threadIdx.x;
  const int g0 = g.layer_goff[l], ng = g.layer_goff[l + 1] - g0;
  extern __shared__ __align__(16) unsigned char smraw[];
  double2* u = reinterpret_cast<double2*>(smraw);       // [ng][y2]: sum over the pads of one x
  for (int i = tid; i < ng * y2; i += 256) {
    const int gi = i / y2, ky = i - gi * y2, grp = g0 + gi;
    double2 s = make_double2(0.0, 0.0);
    for (int p = g.grp_off[grp]; p < g.grp_off[grp + 1]; ++p) {
      const int b = g.grp_pad[p];
      const double2 w = g.twyd[(ky * g.pad_y[b]) % ny];
      const double q = g.q[b];
      s.x += q * w.x; s.y += q * w.y;
    }
    u[i] = s;
  }
  __syncthreads();
  const int kx0 = blockIdx.x * kInjKx;
  for (int i = tid; i < kInjKx * y2; i += 256) {
    const int kx = kx0 + i / y2, ky = i % y2;
    if (kx >= nx) continue;
    double2 a = make_double2(0.0, 0.0);
    for (int gi = 0; gi < ng; ++gi) {
      const double2 p = dmul(u[gi * y2 + ky], g.twxd[(kx * g.grp_x[g0 + gi]) % nx]);
      a.x += p.x; a.y += p.y;
    }
    if (kx == nx / 2) a = make_double2(0.0, 0.0);        // removed Nyquist plane (R11)
    g.qh[((size_t)l * nx + kx) * y2 + ky] = make_float2((float)(a.x * gd.inv_n), (float)(a.y * gd.inv_n));
  }
}

}  // namespace wt
