// Boundary adjust of wt_solve_H (steps a3, a4): the point charges on the pad nodes are "adjusted,
// in magnitude, to enforce the boundary conditions" (R8-R10 exact collocation), fp64.
//
//   phase 1  V_rho at every pad node from the fp64 mixed-space planes pl[l][kx][ky] = V~_rho(kx, z_l, ky)
//            (written by the z-line kernel), evaluated separably: first along kx for each distinct pad
//            x of the layer (a "group"), then along ky per pad;  rhs = flag * V_pad - V_rho|_B
//   phase 2  Q' = Ainv rhs (one warp per row)
//   phase 3  Q^_l(kx,ky) = (1/N) sum_{b in layer l} Q'_b e^{-i(kx x_b + ky y_b)}, separably again (along y
//            per group, then along x); the plane kernel multiplies it with the translated fundamental
//            solution g~(kx, z - z_l, ky)  (the paper's V_ext in O(N) instead of O(|B| N))
//
// k_boundary<0> runs the three phases in ONE launch on a thread-block cluster of kBndCluster CTAs per
// geometry (cluster barriers between the phases; small pad sets: the chain is latency bound);
// k_boundary<1|2|3> run one phase each on as many CTAs as there are work units (large pad sets:
// Ainv is streamed by the whole chip).  Work units are strided over the CTAs of the launch.
#pragma once
#include <cooperative_groups.h>

#include "solve_common.cuh"

namespace wt {

constexpr int kBndCluster = 8;
constexpr int kBndThreads = 512;
constexpr int kBndChunks = 16;   // kx range split of phase 1
constexpr int kBndKx = 16;       // kx values per work unit of phase 3

struct BndSmem {                  // byte offsets into the dynamic shared memory
  size_t twx, twy, work, qs, ys, gx, total;
};
__host__ __device__ inline BndSmem bnd_smem(int nx, int ny, int max_groups_per_layer, int B) {
  BndSmem s;
  const int y2 = ny / 2;
  size_t p = 0;
  s.twx = p; p += (size_t)nx * 16;
  s.twy = p; p += (size_t)ny * 16;
  const size_t w1 = (size_t)(kBndChunks + 1) * y2 * 16, w3 = (size_t)(max_groups_per_layer > 0 ? max_groups_per_layer : 1) * y2 * 16;
  s.work = p; p += (w1 > w3 ? w1 : w3);
  s.qs = p; p += (size_t)(B > 0 ? B : 1) * 8;
  s.ys = p; p += (size_t)(B > 0 ? B : 1) * 4;
  s.gx = p; p += (size_t)(B > 0 ? B : 1) * 4;
  s.total = (p + 15) / 16 * 16;
  return s;
}

// grid (n_cta, n_geoms_in_batch), block kBndThreads.  PHASE 0: n_cta = kBndCluster = one cluster.
template <int PHASE>
__global__ void __launch_bounds__(kBndThreads)
k_boundary(const __grid_constant__ GeomBatch gb, GridDev gd, int max_gl, int substep, int emit, double flag) {
  const GeomDev& g = gb.g[blockIdx.y];
  if (substep >= g.n_sub || g.B == 0) return;       // uniform over the geometry's CTAs
  const int nx = gd.nx, ny = gd.ny, y2 = gd.y2, tid = threadIdx.x;
  const int cta = blockIdx.x, n_cta = gridDim.x;
  const int B = g.B;
  extern __shared__ __align__(16) unsigned char smraw[];
  const BndSmem so = bnd_smem(nx, ny, max_gl, B);
  double2* twx = reinterpret_cast<double2*>(smraw + so.twx);    // e^{-2 pi i k/nx}
  double2* twy = reinterpret_cast<double2*>(smraw + so.twy);
  double2* work = reinterpret_cast<double2*>(smraw + so.work);
  double* qs = reinterpret_cast<double*>(smraw + so.qs);
  int* ys = reinterpret_cast<int*>(smraw + so.ys);      // y of pad i
  int* gx = reinterpret_cast<int*>(smraw + so.gx);      // x of group k
  const int warp = tid >> 5, lane = tid & 31;
  constexpr int kWarps = kBndThreads / 32;

  if (PHASE != 2) {
    for (int i = tid; i < nx; i += kBndThreads) twx[i] = g.twxd[i];
    for (int i = tid; i < ny; i += kBndThreads) twy[i] = g.twyd[i];
    for (int i = tid; i < B; i += kBndThreads) ys[i] = g.pad_y[i];
    for (int i = tid; i < g.G; i += kBndThreads) gx[i] = g.grp_x[i];
    __syncthreads();
  }

  // ---- phase 1: pad potentials of the free charge ------------------------------------------------
  if (PHASE == 0 || PHASE == 1) {
    double2* part = work;                               // [kBndChunks][y2]
    double2* tl = work + kBndChunks * y2;               // [y2]
    const int per = (nx + kBndChunks - 1) / kBndChunks;
    for (int grp = cta; grp < g.G; grp += n_cta) {
      const int l = g.grp_layer[grp], x = gx[grp];
      const int p0 = g.grp_off[grp], p1 = g.grp_off[grp + 1];
      const double2* __restrict__ pl = (emit ? g.pl_e : g.pl) + (size_t)l * nx * y2;
      for (int i = tid; i < y2 * kBndChunks; i += kBndThreads) {
        const int ky = i % y2, ch = i / y2;
        const int k0 = ch * per, k1 = min(nx, k0 + per);
        double2 s = make_double2(0.0, 0.0);
        for (int kx = k0; kx < k1; ++kx) {
          double2 w = twx[(kx * x) % nx];
          w.y = -w.y;                                   // e^{+i kx x}
          const double2 p = dmul(pl[(size_t)kx * y2 + ky], w);
          s.x += p.x; s.y += p.y;
        }
        part[ch * y2 + ky] = s;
      }
      __syncthreads();
      for (int ky = tid; ky < y2; ky += kBndThreads) {
        double2 s = make_double2(0.0, 0.0);
#pragma unroll
        for (int ch = 0; ch < kBndChunks; ++ch) { const double2 p = part[ch * y2 + ky]; s.x += p.x; s.y += p.y; }
        const double wgt = (ky == 0) ? 1.0 : 2.0;       // Hermitian half spectrum along y
        tl[ky] = make_double2(wgt * s.x, wgt * s.y);
      }
      __syncthreads();
      for (int i = p0 + warp; i < p1; i += kWarps) {
        const int y = ys[i];
        double s = 0.0;
        for (int ky = lane; ky < y2; ky += 32) {
          const double2 w = twy[(ky * y) % ny];         // Re(T e^{+i ky y}) = T.x w.x + T.y w.y, w = e^{-i ky y}
          const double2 t = tl[ky];
          s += t.x * w.x + t.y * w.y;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) g.rhs[i] = flag * g.pad_pot[i] - s;
      }
      __syncthreads();                                  // part / tl are reused by the next group
    }
  }
  if (PHASE == 0) cooperative_groups::this_cluster().sync();

  // ---- phase 2: Q' = Ainv rhs ----------------------------------------------------------------------
  if (PHASE == 0 || PHASE == 2) {
    for (int row = cta * kWarps + warp; row < B; row += n_cta * kWarps) {
      const double* __restrict__ a = g.ainv + (size_t)row * B;
      double s = 0.0;
      for (int jj = lane; jj < B; jj += 32) s += a[jj] * __ldcg(g.rhs + jj);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (lane == 0) g.q[row] = s;
    }
  }
  if (PHASE == 0) cooperative_groups::this_cluster().sync();

  // ---- phase 3: spectrum of the boundary charges per pad layer -------------------------------------
  if (PHASE == 0 || PHASE == 3) {
    for (int i = tid; i < B; i += kBndThreads) qs[i] = __ldcg(g.q + i);
    __syncthreads();
    const int kchunks = (nx + kBndKx - 1) / kBndKx;
    int l_have = -1;
    double2* u = work;                                  // [groups of the layer][y2]
    for (int unit = cta; unit < g.L * kchunks; unit += n_cta) {
      const int l = unit / kchunks, kx0 = (unit - l * kchunks) * kBndKx;
      const int g0 = g.layer_goff[l], ng = g.layer_goff[l + 1] - g0;
      if (l != l_have) {
        __syncthreads();
        for (int i = tid; i < ng * y2; i += kBndThreads) {
          const int gi = i / y2, ky = i - gi * y2, grp = g0 + gi;
          double2 s = make_double2(0.0, 0.0);
          const int p0 = g.grp_off[grp], p1 = g.grp_off[grp + 1];
          for (int p = p0; p < p1; ++p) {
            const double2 w = twy[(ky * ys[p]) % ny];
            const double q = qs[p];
            s.x += q * w.x; s.y += q * w.y;
          }
          u[i] = s;
        }
        __syncthreads();
        l_have = l;
      }
      for (int i = tid; i < kBndKx * y2; i += kBndThreads) {
        const int kx = kx0 + i / y2, ky = i % y2;
        if (kx >= nx) continue;
        double2 a = make_double2(0.0, 0.0);
        for (int gi = 0; gi < ng; ++gi) {
          const double2 p = dmul(u[gi * y2 + ky], twx[(kx * gx[g0 + gi]) % nx]);
          a.x += p.x; a.y += p.y;
        }
        if (kx == nx / 2) a = make_double2(0.0, 0.0);   // removed Nyquist plane (R11)
        g.qh[((size_t)l * nx + kx) * y2 + ky] = make_float2((float)(a.x * gd.inv_n), (float)(a.y * gd.inv_n));
      }
    }
  }
}

}  // namespace wt
