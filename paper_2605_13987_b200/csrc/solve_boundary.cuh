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
// k_boundary_cluster runs the three phases in ONE launch on a thread-block cluster of kBndCluster CTAs
// per geometry (small pad sets: the chain is latency bound);
// k_boundary<1|2> + k_boundary_qh run one phase each on as many CTAs as there are work units (large pad sets:
// Ainv is streamed by the whole chip).  Work units are strided over the CTAs of the launch.
#pragma once
#include <cooperative_groups.h>
#include <cuda_pipeline.h>

#include "fft.cuh"
#include "solve_common.cuh"

namespace wt {

// clock stamps of thread 0 of each CTA of geometry 0: only in -DWTIDE_DEBUG builds (never in the shipped library)
#ifdef WTIDE_DEBUG
#define WT_STAMP(k) do { if (gd.stamps && threadIdx.x == 0 && blockIdx.y == 0) gd.stamps[blockIdx.x * 16 + (k)] = clock64(); } while (0)
#else
#define WT_STAMP(k) do { } while (0)
#endif

constexpr int kBndCluster = 8;
constexpr int kBndThreads = 512;
constexpr int kBndChunks = 16;   // kx range split of phase 1

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

// grid (n_cta, n_geoms_in_batch), block kBndThreads.
// NXY: compile-time plane size (nx = ny = NXY; 0 = run-time sizes)
template <int PHASE, int NXY = 0>
__global__ void __launch_bounds__(kBndThreads)
k_boundary(const __grid_constant__ GeomBatch gb, GridDev gd, int max_gl, int substep, int emit, double flag) {
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.y];
  if (substep >= g.n_sub || g.B == 0) { pdl_wait(); return; }   // uniform over the geometry's CTAs
  pdl_wait();
  const int nx = NXY ? NXY : gd.nx, ny = NXY ? NXY : gd.ny, y2 = ny / 2, tid = threadIdx.x;
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
  if (PHASE == 1) {
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
  // ---- phase 2: Q' = Ainv rhs ----------------------------------------------------------------------
  if (PHASE == 2) {
    // rhs once into shared memory; a warp per row, 16-byte loads, four independent partial sums per lane (fixed order)
    for (int i = tid; i < B; i += kBndThreads) qs[i] = __ldcg(g.rhs + i);
    __syncthreads();
    const int n2 = B >> 1;
    for (int row = cta * kWarps + warp; row < B; row += n_cta * kWarps) {
      const double* __restrict__ a = g.ainv + (size_t)row * g.Bs;            // rows are 16-byte aligned (Bs even)
      const double2* __restrict__ a2 = reinterpret_cast<const double2*>(a);
      double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
      for (int jj = lane; jj < n2; jj += 64) {
        const double2 v = a2[jj];
        const bool more = jj + 32 < n2;
        const double2 u = more ? a2[jj + 32] : make_double2(0.0, 0.0);
        s0 = fma(v.x, qs[2 * jj], s0); s1 = fma(v.y, qs[2 * jj + 1], s1);
        if (more) { s2 = fma(u.x, qs[2 * jj + 64], s2); s3 = fma(u.y, qs[2 * jj + 65], s3); }
      }
      if ((B & 1) && lane == 0) s0 = fma(a[B - 1], qs[B - 1], s0);
      double sum = (s0 + s1) + (s2 + s3);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
      if (lane == 0) g.q[row] = sum;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// k_boundary_qh (phase 3 of the split boundary adjust): spectrum of the boundary point charges of one pad layer,
//   qh[l][kx][ky] = (1/N) sum_{b in layer l} Q'_b e^{-i (kx x_b + ky y_b)},  ky < ny/2, 0 at kx = nx/2 (R11),
// as ONE real 2-D transform of the layer's charge image in shared memory (two x-rows packed into a complex line, as in
// k_plane) instead of a sum over the pads per mode: its cost does not grow with the pad count.  fp32: it feeds the fp32
// fields (the persistent solver forms the same spectrum in fp32).  grid (L, n_geoms), block kBndThreads,
// dynamic smem (2 (nx/2)(ny+1) + nx + ny) float2 + (2 nx + 1) ints.
// ------------------------------------------------------------------------------------------------
// NXY: compile-time plane size (nx = ny = NXY; 0 = run-time sizes): the index arithmetic of the passes folds to constants
template <int NXY>
__global__ void __launch_bounds__(kBndThreads)
k_boundary_qh(const __grid_constant__ GeomBatch gb, GridDev gd, int substep) {
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.y];
  const int l = blockIdx.x;
  if (substep >= g.n_sub || g.B == 0 || l >= g.L) { pdl_wait(); return; }
  const int nx = NXY ? NXY : gd.nx, ny = NXY ? NXY : gd.ny, y2 = ny / 2, hx = nx / 2, nyp = ny + 1;
  const int tid = threadIdx.x, bd = blockDim.x;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* w1 = reinterpret_cast<float2*>(smraw);
  float2* w2 = w1 + (size_t)hx * nyp;
  float2* s_twx = w2 + (size_t)hx * nyp;
  float2* s_twy = s_twx + nx;
  for (int i = tid; i < nx; i += bd) s_twx[i] = g.twx[i];
  for (int i = tid; i < ny; i += bd) s_twy[i] = g.twy[i];
  for (int i = tid; i < hx * nyp; i += bd) w1[i] = make_float2(0.f, 0.f);
  int* s_goff = reinterpret_cast<int*>(s_twy + ny);      // [ng + 1] pad offsets of the layer's groups (static tables: before the wait)
  int* s_gx = s_goff + (g.lgoff[l + 1] - g.lgoff[l]) + 1;   // [ng]
  for (int i = tid; i <= g.lgoff[l + 1] - g.lgoff[l]; i += bd) s_goff[i] = g.grp_off[g.lgoff[l] + i];
  for (int i = tid; i < g.lgoff[l + 1] - g.lgoff[l]; i += bd) s_gx[i] = g.grp_x[g.lgoff[l] + i];
  __syncthreads();
  pdl_wait();
  // the layer's charge image: pad (x, y) -> line x/2, real part for even x, imaginary part for odd x (each node holds one pad)
  // (one thread per pad: its group, hence its x, by bisection of the layer's group offsets held in shared memory)
  float* img = reinterpret_cast<float*>(w1);
  {
    const int g0 = g.lgoff[l], ng = g.lgoff[l + 1] - g0;
    const int P0 = s_goff[0], P1 = s_goff[ng];
    for (int p = P0 + tid; p < P1; p += bd) {
      int lo = 0, hi = ng - 1;                         // largest k with s_goff[k] <= p
      while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (s_goff[mid] <= p) lo = mid; else hi = mid - 1; }
      const int x = s_gx[lo];
      img[2 * ((x >> 1) * nyp + g.pad_y[p]) + (x & 1)] = (float)(__ldcg(g.q + p) * gd.inv_n);
    }
  }
  __syncthreads();
  float2* jf = fft_lines<float2>(w1, w2, ny, hx, nyp, 1, s_twy, false);
  float2* jo = (jf == w1) ? w2 : w1;
  for (int t = tid; t < hx * y2; t += bd) {
    const int p = t / y2, k = t - p * y2;
    const float2 zk = jf[p * nyp + k];
    const float2 zm = jf[p * nyp + (k == 0 ? 0 : ny - k)];
    jo[(2 * p) * y2 + k] = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
    jo[(2 * p + 1) * y2 + k] = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
  }
  __syncthreads();
  float2* jt = fft_lines<float2>(jo, jf, nx, y2, 1, y2, s_twx, false);
  float2* __restrict__ out = g.qh + (size_t)l * nx * y2;
  for (int t = tid; t < nx * y2; t += bd) out[t] = (t / y2 == nx / 2) ? make_float2(0.f, 0.f) : jt[t];   // removed Nyquist plane (R11)
}


// ------------------------------------------------------------------------------------------------
// k_boundary_cluster: the three phases in ONE launch on a cluster of CL CTAs per geometry (CL = 16
// where the device grants the non-portable size, else 8), written for latency -- the chain
// z-line kernel -> boundary -> plane kernel is serial and the pad sets are small, so what counts is
// the number of dependent steps, not throughput:
//   - the CTA's row slice of Ainv arrives by ONE bulk (TMA) copy, issued first and awaited before
//     phase 2; every small table is staged in shared memory once; the first loads of pl are issued
//     before the first barrier (their addresses come from the parameter space alone);
//   - phase 1: each CTA owns a contiguous range of groups; rhs values are pushed into EVERY CTA's
//     shared memory (DSMEM), so that phase 2 needs no global round trip;
//   - phase 2: each CTA owns a contiguous range of rows of Ainv (one warp per row); Q' is pushed
//     the same way;
//   - phase 3: each CTA owns a contiguous range of (layer, kx) rows of Q^_l.
// Two cluster barriers in total.  Summation orders are fixed (run-to-run deterministic).
// POW2: nx and ny are powers of two (index arithmetic by masks instead of integer division).
// ------------------------------------------------------------------------------------------------
constexpr int kBclThreads = 1024;

struct BndClSmem {
  size_t bar, twx, twy, vpad, rhs, q, work, wtab, ys, gx, gl, goff, ainv, total;
  int kc, gpc, rows, rpc, lcl, in_smem;
};
__host__ __device__ inline BndClSmem bnd_cl_smem(int nx, int ny, int L, int G, int B, int Bs, int CL, bool ainv_in_smem,
                                                 int threads = kBclThreads) {
  BndClSmem s;
  const int y2 = ny / 2;
  const int Gp = G > 0 ? G : 1, Bp = B > 0 ? B : 1, Lp = L > 0 ? L : 1;
  s.lcl = CL == 16 ? 4 : 3;
  s.in_smem = ainv_in_smem ? 1 : 0;
  s.kc = threads / y2 < 1 ? 1 : (threads / y2 > nx ? nx : threads / y2);
  s.gpc = (Gp + CL - 1) / CL;
  s.rows = (Bp + CL - 1) / CL;
  s.rpc = (Lp * nx + CL - 1) / CL;
  size_t p = 0;
  s.bar = p; p += 16;
  s.twx = p; p += (size_t)nx * 16;
  s.twy = p; p += (size_t)ny * 16;
  const size_t w1 = (size_t)(s.kc + 1) * s.gpc * y2 * 16, w3 = ((size_t)Gp + 4 * (size_t)s.rpc) * y2 * 16;
  s.work = p; p += (w1 > w3 ? w1 : w3);
  s.wtab = p; p += (size_t)s.rpc * Gp * 16;
  s.ainv = p; p += ainv_in_smem ? (size_t)s.rows * Bs * 8 : 0;
  s.vpad = p; p += (size_t)Bp * 8;
  s.rhs = p; p += (size_t)Bp * 8;
  s.q = p; p += (size_t)Bp * 8;
  s.ys = p; p += (size_t)Bp * 4;
  s.gx = p; p += (size_t)Gp * 4;
  s.gl = p; p += (size_t)Gp * 4;
  s.goff = p; p += (size_t)(Gp + 1) * 4;
  s.total = (p + 15) / 16 * 16;
  return s;
}

template <bool POW2>
__global__ void __launch_bounds__(kBclThreads, 1)
k_boundary_cluster(const __grid_constant__ GeomBatch gb, GridDev gd, int max_g, int max_b, int max_bs, int ainv_in_smem,
                   int substep, int emit, double flag) {
  namespace cg = cooperative_groups;
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.y];
  if (substep >= g.n_sub || g.B == 0) { pdl_wait(); return; }   // uniform over the cluster
  pdl_wait();
  cg::cluster_group cluster = cg::this_cluster();
  cluster.barrier_arrive();                         // (waited for before the first remote store)
  WT_STAMP(0);
  const int CL = gridDim.x;                         // grid.x == cluster size
  const int rank = blockIdx.x;
  const int nx = gd.nx, ny = gd.ny, y2 = gd.y2, tid = threadIdx.x;
  const int B = g.B, Bs = g.Bs, G = g.G, L = g.L;
  auto modx = [&](int v) { return POW2 ? (v & (nx - 1)) : (v % nx); };
  auto mody = [&](int v) { return POW2 ? (v & (ny - 1)) : (v % ny); };
  extern __shared__ __align__(16) unsigned char smraw[];
  const BndClSmem so = bnd_cl_smem(nx, ny, kMaxLayers, max_g, max_b, max_bs, CL, ainv_in_smem != 0);
  double2* twx = reinterpret_cast<double2*>(smraw + so.twx);    // e^{-2 pi i k/nx}
  double2* twy = reinterpret_cast<double2*>(smraw + so.twy);
  double2* work = reinterpret_cast<double2*>(smraw + so.work);
  double2* wtab = reinterpret_cast<double2*>(smraw + so.wtab);
  double* vpad = reinterpret_cast<double*>(smraw + so.vpad);
  double* rhs = reinterpret_cast<double*>(smraw + so.rhs);
  double* qs = reinterpret_cast<double*>(smraw + so.q);
  double* As = reinterpret_cast<double*>(smraw + so.ainv);
  int* ys = reinterpret_cast<int*>(smraw + so.ys);
  int* gx = reinterpret_cast<int*>(smraw + so.gx);
  int* gl = reinterpret_cast<int*>(smraw + so.gl);
  int* goff = reinterpret_cast<int*>(smraw + so.goff);
  const int warp = tid >> 5, lane = tid & 31;
  constexpr int kWarps = kBclThreads / 32;

  // rows of Ainv this CTA owns: one bulk copy global -> shared, completion on an mbarrier
  const int rows_per = (B + CL - 1) / CL;
  const int r0 = min(B, rank * rows_per), r1 = min(B, r0 + rows_per);
  const bool bulk = ainv_in_smem && r1 > r0;
  const unsigned bar = (unsigned)__cvta_generic_to_shared(smraw + so.bar);
  if (bulk && tid == 0) {
    const unsigned bytes = (unsigned)(r1 - r0) * (unsigned)Bs * 8u;
    const unsigned dst = (unsigned)__cvta_generic_to_shared(As);
    const double* src = g.ainv + (size_t)r0 * Bs;
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
  }
  for (int i = tid; i < nx; i += kBclThreads) twx[i] = g.twxd[i];
  for (int i = tid; i < ny; i += kBclThreads) twy[i] = g.twyd[i];
  for (int i = tid; i < B; i += kBclThreads) { ys[i] = g.pad_y[i]; vpad[i] = g.pad_pot[i]; }
  for (int i = tid; i < G; i += kBclThreads) { gx[i] = g.grp_x[i]; gl[i] = g.grp_layer[i]; }
  for (int i = tid; i <= G; i += kBclThreads) goff[i] = g.grp_off[i];

  // ---- phase 1: pad potentials of the free charge, groups [gbeg, gbeg + ng) ------------------------
  {
    const int gpc = (G + CL - 1) / CL;
    const int gbeg = min(G, rank * gpc), ng = min(G, gbeg + gpc) - gbeg;
    const int KC = so.kc, per = (nx + KC - 1) / KC;
    double2* part = work;                               // [ng][KC][y2]
    double2* tl = work + (size_t)so.gpc * KC * y2;      // [ng][y2]
    const double2* __restrict__ plb = emit ? g.pl_e : g.pl;
    // the first loads of pl need no table: the layer of group gbeg follows from the parameter space
    constexpr int kPre = 4;                             // kx values held in registers
    const bool one_pass = (KC * y2 <= kBclThreads) && per <= kPre && ng > 0;
    double2 pre[kPre];
    int pre_layer = 0;
#pragma unroll
    for (int l = 1; l < kMaxLayers; ++l) pre_layer += (l < L && g.lgoff[l] <= gbeg) ? 1 : 0;
    if (one_pass && tid < KC * y2) {
      const int ky = tid % y2, ch = tid / y2, k0 = min(nx, ch * per);
#pragma unroll
      for (int r = 0; r < kPre; ++r)
        pre[r] = (k0 + r < nx && r < per) ? plb[((size_t)pre_layer * nx + k0 + r) * y2 + ky] : make_double2(0.0, 0.0);
    }
    WT_STAMP(1);
    __syncthreads();
    WT_STAMP(2);
    for (int i = tid; i < KC * y2; i += kBclThreads) {
      const int ky = i % y2, ch = i / y2;
      const int k0 = min(nx, ch * per), k1 = min(nx, k0 + per);
      for (int gi = 0; gi < ng; ++gi) {
        const int x = gx[gbeg + gi], l = gl[gbeg + gi];
        int idx = modx(k0 * x);
        double2 s = make_double2(0.0, 0.0);
        if (one_pass && l == pre_layer) {
#pragma unroll
          for (int r = 0; r < kPre; ++r) {
            if (k0 + r < k1) {
              double2 w = twx[idx];
              w.y = -w.y;                               // e^{+i kx x}
              const double2 p = dmul(pre[r], w);
              s.x += p.x; s.y += p.y;
              idx += x; if (idx >= nx) idx -= nx;
            }
          }
        } else {
          const double2* __restrict__ pl = plb + (size_t)l * nx * y2 + ky;
          for (int kx = k0; kx < k1; ++kx) {
            double2 w = twx[idx];
            w.y = -w.y;
            const double2 p = dmul(pl[(size_t)kx * y2], w);
            s.x += p.x; s.y += p.y;
            idx += x; if (idx >= nx) idx -= nx;
          }
        }
        part[((size_t)gi * KC + ch) * y2 + ky] = s;
      }
    }
    __syncthreads();
    WT_STAMP(3);
    for (int i = tid; i < ng * y2; i += kBclThreads) {
      const int gi = i / y2, ky = i - gi * y2;
      const double2* __restrict__ pp = part + (size_t)gi * KC * y2 + ky;
      double2 s = make_double2(0.0, 0.0);
#pragma unroll 8
      for (int ch = 0; ch < KC; ++ch) { const double2 p = pp[ch * y2]; s.x += p.x; s.y += p.y; }
      const double wgt = (ky == 0) ? 1.0 : 2.0;         // Hermitian half spectrum along y
      tl[i] = make_double2(wgt * s.x, wgt * s.y);
    }
    __syncthreads();
    WT_STAMP(4);
    cluster.barrier_wait();                             // every CTA of the cluster is running
    const int pbeg = goff[gbeg], pend = goff[gbeg + ng];
    for (int p = pbeg + warp; p < pend; p += kWarps) {
      int gi = 0;
      while (goff[gbeg + gi + 1] <= p) ++gi;
      const int y = ys[p];
      double s = 0.0;
      for (int ky = lane; ky < y2; ky += 32) {
        const double2 w = twy[mody(ky * y)];            // Re(T e^{+i ky y}) = T.x w.x + T.y w.y, w = e^{-i ky y}
        const double2 t = tl[gi * y2 + ky];
        s += t.x * w.x + t.y * w.y;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (lane < CL) cluster.map_shared_rank(rhs, lane)[p] = flag * vpad[p] - s;
    }
  }
  WT_STAMP(5);
  if (bulk) {                                           // the slice of Ainv has landed
    unsigned done = 0;
    while (!done) {
      asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                   : "=r"(done) : "r"(bar), "r"(0u) : "memory");
    }
  }
  WT_STAMP(6);
  cluster.sync();
  WT_STAMP(7);

  // ---- phase 2: Q' = Ainv rhs, rows [r0, r1) ---------------------------------------------------------
  for (int row = r0 + warp; row < r1; row += kWarps) {
    const double* __restrict__ a = ainv_in_smem ? As + (size_t)(row - r0) * Bs : g.ainv + (size_t)row * Bs;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int jj = lane;
    for (; jj + 96 < B; jj += 128) {
      s0 += a[jj] * rhs[jj]; s1 += a[jj + 32] * rhs[jj + 32];
      s2 += a[jj + 64] * rhs[jj + 64]; s3 += a[jj + 96] * rhs[jj + 96];
    }
    for (; jj < B; jj += 32) s0 += a[jj] * rhs[jj];
    double s = (s0 + s1) + (s2 + s3);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane < CL) cluster.map_shared_rank(qs, lane)[row] = s;
  }
  WT_STAMP(8);
  cluster.sync();
  WT_STAMP(9);

  // ---- phase 3: spectrum of the boundary charges, rows (l, kx) in [rw0, rw1) -------------------------
  {
    const int n_rows = L * nx, rpc = (n_rows + CL - 1) / CL;
    const int rw0 = min(n_rows, rank * rpc), rw1 = min(n_rows, rw0 + rpc);
    if (rw0 < rw1) {
      const int l0 = rw0 / nx, l1 = (rw1 - 1) / nx;
      const int ga = g.lgoff[l0], gz = g.lgoff[l1 + 1];
      double2* u = work;                                // [G][y2], groups [ga, gz) filled
      for (int i = ga * y2 + tid; i < gz * y2; i += kBclThreads) {
        const int grp = i / y2, ky = i - grp * y2;
        double2 s0 = make_double2(0.0, 0.0), s1 = make_double2(0.0, 0.0);
        int p = goff[grp];
        const int pe = goff[grp + 1];
        for (; p + 1 < pe; p += 2) {
          const double2 w0 = twy[mody(ky * ys[p])], w1 = twy[mody(ky * ys[p + 1])];
          const double q0 = qs[p], q1 = qs[p + 1];
          s0.x += q0 * w0.x; s0.y += q0 * w0.y;
          s1.x += q1 * w1.x; s1.y += q1 * w1.y;
        }
        if (p < pe) {
          const double2 w0 = twy[mody(ky * ys[p])];
          const double q0 = qs[p];
          s0.x += q0 * w0.x; s0.y += q0 * w0.y;
        }
        u[i] = make_double2(s0.x + s1.x, s0.y + s1.y);
      }
      // wtab[row - rw0][grp] = e^{-i kx x_grp} for the groups of the row's layer
      for (int i = tid; i < (rw1 - rw0) * G; i += kBclThreads) {
        const int r = i / G, grp = i - r * G;
        const int row = rw0 + r, l = row / nx, kx = row - l * nx;
        if (grp >= g.lgoff[l] && grp < g.lgoff[l + 1]) wtab[i] = twx[modx(kx * gx[grp])];
      }
      WT_STAMP(10);
      __syncthreads();
      WT_STAMP(11);
      for (int i = rw0 * y2 + tid; i < rw1 * y2; i += kBclThreads) {
        const int ky = i % y2, row = i / y2, l = row / nx, kx = row - l * nx;
        const double2* __restrict__ wt_ = wtab + (size_t)(row - rw0) * G;
        double2 a0 = make_double2(0.0, 0.0), a1 = make_double2(0.0, 0.0);
        int grp = g.lgoff[l];
        const int ge = g.lgoff[l + 1];
        for (; grp + 1 < ge; grp += 2) {
          const double2 p0 = dmul(u[grp * y2 + ky], wt_[grp]), p1 = dmul(u[(grp + 1) * y2 + ky], wt_[grp + 1]);
          a0.x += p0.x; a0.y += p0.y; a1.x += p1.x; a1.y += p1.y;
        }
        if (grp < ge) { const double2 p0 = dmul(u[grp * y2 + ky], wt_[grp]); a0.x += p0.x; a0.y += p0.y; }
        double2 a = make_double2(a0.x + a1.x, a0.y + a1.y);
        if (kx == nx / 2) a = make_double2(0.0, 0.0);   // removed Nyquist plane (R11)
        g.qh[i] = make_float2((float)(a.x * gd.inv_n), (float)(a.y * gd.inv_n));
      }
    }
  }
  WT_STAMP(12);
}


// ------------------------------------------------------------------------------------------------
// k_boundary_fast<LNX, LY2>: k_boundary_cluster for nx = 2^LNX, ny = 2^(LY2+1) with every index
// operation a shift or a mask and the shared-memory layout computed on the host (the generic kernel
// spends most of its issue slots on integer division).  512 threads.
// ------------------------------------------------------------------------------------------------
constexpr int kBfThreads = 512;

template <int LNX, int LY2>
__global__ void __launch_bounds__(kBfThreads, 1)
k_boundary_fast(const __grid_constant__ GeomBatch gb, GridDev gd, const __grid_constant__ BndClSmem so, int substep, int emit,
                double flag) {
  namespace cg = cooperative_groups;
  constexpr int NX = 1 << LNX, Y2 = 1 << LY2, NY = 2 * Y2;
  constexpr int KC = (kBfThreads / Y2 > NX) ? NX : kBfThreads / Y2;   // kx chunks of phase 1
  constexpr int PER = NX / KC;
  constexpr int kWarps = kBfThreads / 32;
  static_assert(KC * Y2 <= kBfThreads && NX <= kBfThreads && NY <= kBfThreads, "sizes");
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.y];
  if (substep >= g.n_sub || g.B == 0) { pdl_wait(); return; }   // uniform over the cluster
  cg::cluster_group cluster = cg::this_cluster();
  cluster.barrier_arrive();                         // (waited for before the first remote store)
  WT_STAMP(0);
  const int CL = gridDim.x, lcl = so.lcl;           // grid.x == cluster size = 2^lcl
  const int rank = blockIdx.x, tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  const int B = g.B, Bs = g.Bs, G = g.G, L = g.L;
  extern __shared__ __align__(16) unsigned char smraw[];
  double2* twx = reinterpret_cast<double2*>(smraw + so.twx);    // e^{-2 pi i k/nx}
  double2* twy = reinterpret_cast<double2*>(smraw + so.twy);
  double2* work = reinterpret_cast<double2*>(smraw + so.work);
  double2* wtab = reinterpret_cast<double2*>(smraw + so.wtab);
  double* vpad = reinterpret_cast<double*>(smraw + so.vpad);
  double* rhs = reinterpret_cast<double*>(smraw + so.rhs);
  double* qs = reinterpret_cast<double*>(smraw + so.q);
  double* As = reinterpret_cast<double*>(smraw + so.ainv);
  int* ys = reinterpret_cast<int*>(smraw + so.ys);
  int* gx = reinterpret_cast<int*>(smraw + so.gx);
  int* gl = reinterpret_cast<int*>(smraw + so.gl);
  int* goff = reinterpret_cast<int*>(smraw + so.goff);

  // rows of Ainv this CTA owns: one bulk copy global -> shared, completion on an mbarrier
  const int rows_per = (B + CL - 1) >> lcl;
  const int r0 = min(B, rank * rows_per), r1 = min(B, r0 + rows_per);
  const bool bulk = so.in_smem && r1 > r0;
  const unsigned bar = (unsigned)__cvta_generic_to_shared(smraw + so.bar);
  if (bulk && tid == 0) {
    const unsigned bytes = (unsigned)(r1 - r0) * (unsigned)Bs * 8u;
    const unsigned dst = (unsigned)__cvta_generic_to_shared(As);
    const double* src = g.ainv + (size_t)r0 * Bs;
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
  }
  if (tid < NX) twx[tid] = g.twxd[tid];
  if (tid < NY) twy[tid] = g.twyd[tid];
  for (int i = tid; i < B; i += kBfThreads) { ys[i] = g.pad_y[i]; vpad[i] = g.pad_pot[i]; }
  for (int i = tid; i < G; i += kBfThreads) { gx[i] = g.grp_x[i]; gl[i] = g.grp_layer[i]; }
  for (int i = tid; i <= G; i += kBfThreads) goff[i] = g.grp_off[i];

  // rows (l, kx) of Q^ this CTA owns in phase 3
  const int n_rows = L << LNX, rpc = (n_rows + CL - 1) >> lcl;
  const int rw0 = min(n_rows, rank * rpc), rw1 = min(n_rows, rw0 + rpc);
  const int gpc = (G + CL - 1) >> lcl;

  // ---- phase 1: pad potentials of the free charge, groups [gbeg, gbeg + ng) ------------------------
  {
    const int gbeg = min(G, rank * gpc), ng = min(G, gbeg + gpc) - gbeg;
    double2* part = work;                               // [ng][KC][Y2]
    double2* tl = work + (size_t)so.gpc * KC * Y2;      // [ng][Y2]
    const double2* __restrict__ plb = emit ? g.pl_e : g.pl;
    const int ky = tid & (Y2 - 1), ch = tid >> LY2, k0 = ch * PER;
    const bool act = tid < KC * Y2;
    // the first loads of pl need no table: the layer of group gbeg follows from the parameter space
    constexpr int kPre = PER <= 4 ? PER : 1;
    constexpr bool kUsePre = PER <= 4;
    double2 pre[kPre];
    int pre_layer = 0;
#pragma unroll
    for (int l = 1; l < kMaxLayers; ++l) pre_layer += (l < L && g.lgoff[l] <= gbeg) ? 1 : 0;
    pdl_wait();                                         // pl is written by the z-line kernel
    if (kUsePre && act && ng > 0) {
#pragma unroll
      for (int r = 0; r < kPre; ++r) pre[r] = plb[((size_t)pre_layer * NX + k0 + r) * Y2 + ky];
    }
    WT_STAMP(1);
    __syncthreads();
    WT_STAMP(2);
    if (act) {
      for (int gi = 0; gi < ng; ++gi) {
        const int x = gx[gbeg + gi], l = gl[gbeg + gi];
        int idx = (k0 * x) & (NX - 1);
        double2 s = make_double2(0.0, 0.0);
        if (kUsePre && l == pre_layer) {
#pragma unroll
          for (int r = 0; r < kPre; ++r) {
            double2 w = twx[idx];
            w.y = -w.y;                                 // e^{+i kx x}
            const double2 p = dmul(pre[r], w);
            s.x += p.x; s.y += p.y;
            idx = (idx + x) & (NX - 1);
          }
        } else {
          const double2* __restrict__ pl = plb + ((size_t)l * NX + k0) * Y2 + ky;
#pragma unroll 4
          for (int r = 0; r < PER; ++r) {
            double2 w = twx[idx];
            w.y = -w.y;
            const double2 p = dmul(pl[(size_t)r * Y2], w);
            s.x += p.x; s.y += p.y;
            idx = (idx + x) & (NX - 1);
          }
        }
        part[(gi * KC + ch) * Y2 + ky] = s;
      }
    }
    // (independent of the charges) wtab[row - rw0][grp] = e^{-i kx x_grp} for phase 3
    for (int r = warp; r < rw1 - rw0; r += kWarps) {
      const int row = rw0 + r, l = row >> LNX, kx = row & (NX - 1);
      for (int grp = g.lgoff[l] + lane; grp < g.lgoff[l + 1]; grp += 32) wtab[r * G + grp] = twx[(kx * gx[grp]) & (NX - 1)];
    }
    __syncthreads();
    WT_STAMP(3);
    for (int i = tid; i < ng * Y2; i += kBfThreads) {
      const int gi = i >> LY2, kk = i & (Y2 - 1);
      const double2* __restrict__ pp = part + gi * KC * Y2 + kk;
      double2 s0 = make_double2(0.0, 0.0), s1 = make_double2(0.0, 0.0);
#pragma unroll
      for (int c = 0; c < KC; c += 2) {
        const double2 p = pp[c * Y2];
        s0.x += p.x; s0.y += p.y;
        if (c + 1 < KC) { const double2 q = pp[(c + 1) * Y2]; s1.x += q.x; s1.y += q.y; }
      }
      const double wgt = (kk == 0) ? 1.0 : 2.0;         // Hermitian half spectrum along y
      tl[i] = make_double2(wgt * (s0.x + s1.x), wgt * (s0.y + s1.y));
    }
    __syncthreads();
    WT_STAMP(4);
    cluster.barrier_wait();                             // every CTA of the cluster is running
    const int pbeg = goff[gbeg], pend = goff[gbeg + ng];
    for (int p = pbeg + warp; p < pend; p += kWarps) {
      int gi = 0;
      while (goff[gbeg + gi + 1] <= p) ++gi;
      const int y = ys[p];
      double s = 0.0;
#pragma unroll
      for (int kk = lane; kk < Y2; kk += 32) {
        const double2 w = twy[(kk * y) & (NY - 1)];     // Re(T e^{+i ky y}) = T.x w.x + T.y w.y, w = e^{-i ky y}
        const double2 t = tl[gi * Y2 + kk];
        s += t.x * w.x + t.y * w.y;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (lane == 0) rhs[p] = flag * vpad[p] - s;
    }
  }
  WT_STAMP(5);
  if (bulk) {                                           // the slice of Ainv has landed
    unsigned done = 0;
    while (!done) {
      asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                   : "=r"(done) : "r"(bar), "r"(0u) : "memory");
    }
  }
  WT_STAMP(6);
  cluster.sync();
  WT_STAMP(7);
  // pull the other CTAs' rhs values (one warp per remote CTA, coalesced DSMEM reads)
  for (int r = warp; r < CL; r += kWarps) {
    if (r == rank) continue;
    const int gb0 = min(G, r * gpc), gb1 = min(G, gb0 + gpc);
    const double* __restrict__ remote = cluster.map_shared_rank(rhs, r);
    for (int p = goff[gb0] + lane; p < goff[gb1]; p += 32) rhs[p] = remote[p];
  }
  __syncthreads();

  // ---- phase 2: Q' = Ainv rhs, rows [r0, r1) ---------------------------------------------------------
  for (int row = r0 + warp; row < r1; row += kWarps) {
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int jj = lane;
    if (so.in_smem) {
      const double* __restrict__ a = As + (row - r0) * Bs;
      for (; jj + 96 < B; jj += 128) {
        s0 += a[jj] * rhs[jj]; s1 += a[jj + 32] * rhs[jj + 32];
        s2 += a[jj + 64] * rhs[jj + 64]; s3 += a[jj + 96] * rhs[jj + 96];
      }
      for (; jj < B; jj += 32) s0 += a[jj] * rhs[jj];
    } else {
      const double* __restrict__ a = g.ainv + (size_t)row * Bs;
      for (; jj + 96 < B; jj += 128) {
        s0 += a[jj] * rhs[jj]; s1 += a[jj + 32] * rhs[jj + 32];
        s2 += a[jj + 64] * rhs[jj + 64]; s3 += a[jj + 96] * rhs[jj + 96];
      }
      for (; jj < B; jj += 32) s0 += a[jj] * rhs[jj];
    }
    double s = (s0 + s1) + (s2 + s3);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) qs[row] = s;
  }
  WT_STAMP(8);
  cluster.sync();
  WT_STAMP(9);
  for (int r = warp; r < CL; r += kWarps) {
    if (r == rank) continue;
    const int q0 = min(B, r * rows_per), q1 = min(B, q0 + rows_per);
    const double* __restrict__ remote = cluster.map_shared_rank(qs, r);
    for (int p = q0 + lane; p < q1; p += 32) qs[p] = remote[p];
  }
  cluster.barrier_arrive();                             // (no remote access after this point; waited for at exit)
  __syncthreads();

  // ---- phase 3: spectrum of the boundary charges, rows (l, kx) in [rw0, rw1) -------------------------
  if (rw0 < rw1) {
    const int l0 = rw0 >> LNX, l1 = (rw1 - 1) >> LNX;
    const int ga = g.lgoff[l0], gz = g.lgoff[l1 + 1];
    double2* u = work;                                  // [G][Y2], groups [ga, gz) filled
    for (int i = ga * Y2 + tid; i < gz * Y2; i += kBfThreads) {
      // u[grp][ky] = sum_p Q'_p e^{-i ky y_p}; along a run of consecutive y the phase advances by the
      // fixed factor e^{-i ky} (one table lookup per run instead of one per pad)
      const int grp = i >> LY2, kk = i & (Y2 - 1);
      const double2 stepw = twy[kk];
      double2 s = make_double2(0.0, 0.0), w = make_double2(1.0, 0.0);
      int yprev = -2;
      for (int p = goff[grp]; p < goff[grp + 1]; ++p) {
        const int y = ys[p];
        w = (y == yprev + 1) ? dmul(w, stepw) : twy[(kk * y) & (NY - 1)];
        yprev = y;
        const double q = qs[p];
        s.x += q * w.x; s.y += q * w.y;
      }
      u[i] = s;
    }
    WT_STAMP(10);
    __syncthreads();
    WT_STAMP(11);
    // Q^_l[kx][ky] = (1/N) sum_{g in l} u[g][ky] e^{-i kx x_g}: the group range is split over kSplit thread sets
    const int n_out = (rw1 - rw0) * Y2;
    int kSplit = 1;
    while (kSplit < 4 && n_out * (kSplit * 2) <= kBfThreads) kSplit *= 2;
    double2* red = work + (size_t)G * Y2;               // [kSplit][n_out]  (after u)
    for (int i0 = 0; i0 < n_out; i0 += kBfThreads / kSplit) {
      const int o = i0 + (tid % (kBfThreads / kSplit)), part_i = tid / (kBfThreads / kSplit);
      double2 a0 = make_double2(0.0, 0.0), a1 = make_double2(0.0, 0.0);
      if (o < n_out && part_i < kSplit) {
        const int i = rw0 * Y2 + o;
        const int kk = i & (Y2 - 1), row = i >> LY2, l = row >> LNX;
        const double2* __restrict__ wt_ = wtab + (row - rw0) * G;
        const double2* __restrict__ uu = u + kk;
        const int gs = g.lgoff[l], ge = g.lgoff[l + 1];
        const int per_part = (ge - gs + kSplit - 1) / kSplit;
        int grp = gs + part_i * per_part;
        const int gend = min(ge, grp + per_part);
        for (; grp + 1 < gend; grp += 2) {
          const double2 p0 = dmul(uu[grp * Y2], wt_[grp]), p1 = dmul(uu[(grp + 1) * Y2], wt_[grp + 1]);
          a0.x += p0.x; a0.y += p0.y; a1.x += p1.x; a1.y += p1.y;
        }
        if (grp < gend) { const double2 p0 = dmul(uu[grp * Y2], wt_[grp]); a0.x += p0.x; a0.y += p0.y; }
        red[part_i * n_out + o] = make_double2(a0.x + a1.x, a0.y + a1.y);
      }
      __syncthreads();
      if (o < n_out && part_i == 0) {
        const int i = rw0 * Y2 + o;
        const int kx = (i >> LY2) & (NX - 1);
        double2 a = red[o];
        for (int k = 1; k < kSplit; ++k) { const double2 b = red[k * n_out + o]; a.x += b.x; a.y += b.y; }
        if (kx == NX / 2) a = make_double2(0.0, 0.0);   // removed Nyquist plane (R11)
        g.qh[i] = make_float2((float)(a.x * gd.inv_n), (float)(a.y * gd.inv_n));
      }
      __syncthreads();
    }
  }
  WT_STAMP(12);
  cluster.barrier_wait();
}

}  // namespace wt
