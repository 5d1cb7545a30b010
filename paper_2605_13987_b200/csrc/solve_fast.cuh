// Size-specialised kernels of wt_solve_H for power-of-two grids (the BASELINE configs 0-3):
// register-resident two-stage FFTs (regfft.cuh), all index arithmetic compile-time, one
// __syncthreads per shared-memory exchange.
//
//   k_plane_fast<N, E, CP, EMIT>   xy-plane of an N x N grid, one CTA per z, N*N/(2E) threads;
//                                  CP = 3: the three field components in flight together
//   k_pencil<NZ, E, TYL, ...>      z-lines of length NZ, one CTA per (kx, TYL consecutive ky), TYL*NZ/E threads
//
// Both read/write the mixed-space arrays M[kx][z][ky] of solve_common.cuh exactly like the generic
// kernels (solve_generic.cuh), which remain the path for every other 2^a 3^b size.
#pragma once
#include "regfft.cuh"
#include "solve_common.cuh"

namespace wt {

template <int N> struct PlaneCfg {
  static constexpr int Y2 = N / 2;
  static constexpr int SX = N + 2;       // row stride of the transposed buffer [ky][x] (even: float4 reads)
  static constexpr int SU = N / 2 + 1;   // row stride of the unpack buffer [k][p2] (odd: strided reads conflict free)
  static constexpr int BUF = (Y2 * SX > N * SU) ? Y2 * SX : N * SU;   // float2 per component (>= N*Y2)
};

// ------------------------------------------------------------------------------------------------
// k_plane_fast.  grid (nz, n_geoms), block N*N/(2E), dynamic smem 2 * CP * BUF * 8 bytes.
//
// x-phases: thread (ky = tid % Y2, j = tid / Y2) holds kx (or x) = j + T r, r < E, of line ky.
// y-phases: thread (p2 = tid % Y2, j) holds k (or y) = j + T r of the complex line p2 that packs the
//           real x-rows 2 p2 (real part) and 2 p2 + 1 (imaginary part).
// Exchanges ping-pong between two buffers P and Q: six barriers per component group.
// ------------------------------------------------------------------------------------------------
template <int N, int E, int CP, bool EMIT>
__global__ void __launch_bounds__(N * N / (2 * E), (N <= 64) ? 2 : 1)
k_plane_fast(GridDev gd, const GeomDev* __restrict__ geoms, int substep) {
  using C = PlaneCfg<N>;
  constexpr int Y2 = C::Y2, T = N / E, SX = C::SX, SU = C::SU, BUF = C::BUF;
  static_assert(CP == 1 || CP == 3, "components per group");
  const GeomDev& g = geoms[blockIdx.y];
  if (substep >= g.n_sub) return;
  const int nz = gd.nz, z = blockIdx.x;
  const int tid = threadIdx.x;
  const int ln = tid % Y2;     // line within the phase: ky (x-phases) or p2 (y-phases)
  const int j = tid / Y2;      // position of the thread within its line
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* P = reinterpret_cast<float2*>(smraw);
  float2* Q = P + CP * BUF;
  const float2* __restrict__ mV = EMIT ? g.e0 : g.m0;
  const float2* __restrict__ mE = EMIT ? g.e1 : g.m1;
  const int L = g.L;
  const int slot = EMIT ? (*gd.step % kStageSlots) : 0;

  float2 w[E];
  load_twiddles<E>(w, g.twx, j);          // N x N plane: twx == twy

  // conductivity ids of this thread's nodes in the y-phases: rows 2 ln, 2 ln + 1 at y = j + T r
  unsigned short sid[E];
  if (!EMIT) {
    const unsigned short* st = reinterpret_cast<const unsigned short*>(g.sig_t + (size_t)z * N * N);
#pragma unroll
    for (int r = 0; r < E; ++r) sid[r] = __ldg(st + ((j + T * r) * N + 2 * ln) / 2);
  }
  auto dz_of = [&](int l) { const int d = z - g.layers[l]; return d < 0 ? d + nz : d; };   // (z - z_l) mod nz
  const float kyv = g.kyf[ln];
  float2 dacc[E];                          // D~ = i kx J~x + i ky J~y, accumulated over the components

#pragma unroll
  for (int c0 = 0; c0 < 3; c0 += CP) {
    float2 X[CP][E];
    // ---- load: V~ = V~_rho + sum_l Q^_l g~(z - z_l) (the boundary source, a4); E~ = -i kappa V~ ----------
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int kx = j + T * r;
      const size_t gi = ((size_t)kx * nz + z) * Y2 + ln;
      if constexpr (CP == 3) {
        float2 v = mV[gi], e = mE[gi];
        for (int l = 0; l < L; ++l) {
          const size_t ti = ((size_t)kx * nz + dz_of(l)) * Y2 + ln;
          const float2 qv = g.qh[((size_t)l * N + kx) * Y2 + ln];
          const float gv = __ldg(g.gt + ti), gz = __ldg(g.gzt + ti);
          v.x += qv.x * gv; v.y += qv.y * gv;
          e.x += qv.x * gz; e.y += qv.y * gz;
        }
        const float kxv = g.kxf[kx];
        X[0][r] = make_float2(kxv * v.y, -kxv * v.x);
        X[1][r] = make_float2(kyv * v.y, -kyv * v.x);
        X[2][r] = e;
      } else {
        float2 v = (c0 == 2) ? mE[gi] : mV[gi];
        const float* __restrict__ tab = (c0 == 2) ? g.gzt : g.gt;
        for (int l = 0; l < L; ++l) {
          const float2 qv = g.qh[((size_t)l * N + kx) * Y2 + ln];
          const float gv = __ldg(tab + ((size_t)kx * nz + dz_of(l)) * Y2 + ln);
          v.x += qv.x * gv; v.y += qv.y * gv;
        }
        if (c0 == 0) { const float kxv = g.kxf[kx]; v = make_float2(kxv * v.y, -kxv * v.x); }
        if (c0 == 1) v = make_float2(kyv * v.y, -kyv * v.x);
        X[0][r] = v;
      }
    }
    // ---- A: inverse transform along x ---------------------------------------------------------------
#pragma unroll
    for (int c = 0; c < CP; ++c) {
      fft_stage1<E, true>(X[c], w);
#pragma unroll
      for (int q = 0; q < E; ++q) P[c * BUF + (q * T + j) * Y2 + ln] = X[c][q];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < CP; ++c)
      fft_stage2<E, T, true>(X[c], j, [&](int q, int jj) { return P[c * BUF + (q * T + jj) * Y2 + ln]; });
    // ---- transpose: [ky][x] so that a y-phase thread reads the row pair (2 p2, 2 p2 + 1) as one float4 ---
#pragma unroll
    for (int c = 0; c < CP; ++c)
#pragma unroll
      for (int r = 0; r < E; ++r) Q[c * BUF + ln * SX + j + T * r] = X[c][r];
    __syncthreads();
    // Hermitian completion along y of the two packed real rows (Nyquist = 0): z[k] = a[k] + i b[k]
#pragma unroll
    for (int c = 0; c < CP; ++c)
#pragma unroll
      for (int r = 0; r < E; ++r) {
        if (r < E / 2) {                               // k = j + T r < Y2
          const float4 ab = *reinterpret_cast<const float4*>(&Q[c * BUF + (j + T * r) * SX + 2 * ln]);
          X[c][r] = make_float2(ab.x - ab.w, ab.y + ab.z);
        } else {                                       // k >= Y2: mirror k' = N - k in [1, Y2]
          const int km = N - (j + T * r);
          if (km == Y2) {
            X[c][r] = make_float2(0.f, 0.f);
          } else {
            const float4 ab = *reinterpret_cast<const float4*>(&Q[c * BUF + km * SX + 2 * ln]);
            X[c][r] = make_float2(ab.x + ab.w, ab.z - ab.y);
          }
        }
      }
    // ---- B: inverse transform along y -> E at the nodes (rows 2 ln | 2 ln + 1, y = j + T r) -----------
#pragma unroll
    for (int c = 0; c < CP; ++c) {
      fft_stage1<E, true>(X[c], w);
#pragma unroll
      for (int q = 0; q < E; ++q) P[c * BUF + (q * T + j) * Y2 + ln] = X[c][q];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < CP; ++c)
      fft_stage2<E, T, true>(X[c], j, [&](int q, int jj) { return P[c * BUF + (q * T + jj) * Y2 + ln]; });
    if constexpr (EMIT) {
      // (a8) H[n] = E/dt into the staging slot [slot][comp][z][y][x]
#pragma unroll
      for (int c = 0; c < CP; ++c) {
        float2* st = reinterpret_cast<float2*>(g.stage + (((size_t)slot * 3 + (c0 + c)) * nz + z) * (size_t)(N * N));
#pragma unroll
        for (int r = 0; r < E; ++r)
          st[((j + T * r) * N + 2 * ln) / 2] = make_float2(X[c][r].x * g.inv_dt, X[c][r].y * g.inv_dt);
      }
      if constexpr (CP == 1) __syncthreads();          // P is rewritten by the next component
      continue;
    }
    // ---- conduction current J = (s dt_int) E, nodewise (a6, R17) --------------------------------------
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const float s0 = __ldg(g.sdt + (sid[r] & 0xff)), s1 = __ldg(g.sdt + (sid[r] >> 8));
#pragma unroll
      for (int c = 0; c < CP; ++c) { X[c][r].x *= s0; X[c][r].y *= s1; }
    }
    // ---- C: forward transform along y -----------------------------------------------------------------
#pragma unroll
    for (int c = 0; c < CP; ++c) {
      fft_stage1<E, false>(X[c], w);
#pragma unroll
      for (int q = 0; q < E; ++q) Q[c * BUF + (q * T + j) * Y2 + ln] = X[c][q];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < CP; ++c)
      fft_stage2<E, T, false>(X[c], j, [&](int q, int jj) { return Q[c * BUF + (q * T + jj) * Y2 + ln]; });
    // ---- unpack the two real rows' half spectra: [k][p2], read back with ln = ky ------------------------
#pragma unroll
    for (int c = 0; c < CP; ++c)
#pragma unroll
      for (int r = 0; r < E; ++r) P[c * BUF + (j + T * r) * SU + ln] = X[c][r];
    __syncthreads();
    {
      const int km = (N - ln) % N;
      const bool odd = j & 1;                          // x = j + T r, T even
#pragma unroll
      for (int c = 0; c < CP; ++c)
#pragma unroll
        for (int r = 0; r < E; ++r) {
          const int p2 = (j + T * r) >> 1;
          const float2 zk = P[c * BUF + ln * SU + p2], zm = P[c * BUF + km * SU + p2];
          X[c][r] = odd ? make_float2(0.5f * (zk.y + zm.y), 0.5f * (zm.x - zk.x))
                        : make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
        }
    }
    // ---- D: forward transform along x -----------------------------------------------------------------
#pragma unroll
    for (int c = 0; c < CP; ++c) {
      fft_stage1<E, false>(X[c], w);
#pragma unroll
      for (int q = 0; q < E; ++q) Q[c * BUF + (q * T + j) * Y2 + ln] = X[c][q];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < CP; ++c)
      fft_stage2<E, T, false>(X[c], j, [&](int q, int jj) { return Q[c * BUF + (q * T + jj) * Y2 + ln]; });
    // ---- D~ = i kx J~x + i ky J~y ; J~z goes out as it is ------------------------------------------------
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int kx = j + T * r;
      const size_t gi = ((size_t)kx * nz + z) * Y2 + ln;
      if constexpr (CP == 3) {
        const float kxv = g.kxf[kx];
        const float2 a = X[0][r], b = X[1][r];
        g.m0[gi] = make_float2(-kxv * a.y - kyv * b.y, kxv * a.x + kyv * b.x);
        g.m1[gi] = X[2][r];
      } else {
        const float2 a = X[0][r];
        if (c0 == 0) { const float kxv = g.kxf[kx]; dacc[r] = make_float2(-kxv * a.y, kxv * a.x); }
        if (c0 == 1) { dacc[r].x -= kyv * a.y; dacc[r].y += kyv * a.x; }
        if (c0 == 2) { g.m0[gi] = dacc[r]; g.m1[gi] = a; }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// k_pencil: z-line transforms + per-mode update (a7, a2), pad-layer potentials in fp64 (a3),
// inverse z transforms (a5, z part).  grid (nx * y2/TYL, n_geoms), block TYL * NZ/E.
// Thread (line = tid % TYL, j = tid / TYL) holds z (or kz) = j + T r, r < E, of line ky0 + line.
// dynamic smem: 2 fields * E * QS float2 + L * TYL * T double2.
// ------------------------------------------------------------------------------------------------
template <int NZ, int E, int TYL> struct PencilCfg {
  static constexpr int T = NZ / E;
  static constexpr int PAD = (TYL < 16) ? 16 - TYL : 0;   // skews consecutive q rows across the banks
  static constexpr int QS = T * TYL + PAD;                // float2 per q row of an exchange buffer
  static constexpr int FIELD = E * QS;
  static constexpr int THREADS = T * TYL;
};

// reciprocal of a positive double by Newton iteration from the fp32 estimate (relative error ~1e-16)
__device__ __forceinline__ double fast_rcp(double a) {
  double x = (double)__frcp_rn((float)a);
  x = x * (2.0 - a * x);
  x = x * (2.0 - a * x);
  return x;
}

template <int NZ, int E, int TYL, bool APPLY_J, bool DELTA>
__global__ void __launch_bounds__(PencilCfg<NZ, E, TYL>::THREADS)
k_pencil(GridDev gd, const GeomDev* __restrict__ geoms, int substep, int emit) {
  using C = PencilCfg<NZ, E, TYL>;
  constexpr int T = C::T, QS = C::QS, FIELD = C::FIELD;
  const GeomDev& g = geoms[blockIdx.y];
  if (substep >= g.n_sub) return;
  const int nx = gd.nx, y2 = gd.y2;
  const int tiles = y2 / TYL;
  const int kx = blockIdx.x / tiles, ky0 = (blockIdx.x % tiles) * TYL;
  const int tid = threadIdx.x;
  const int line = tid % TYL, j = tid / TYL;
  const int ky = ky0 + line;
  const int L = g.L;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* buf = reinterpret_cast<float2*>(smraw);                 // [2][E][QS]
  double2* red = reinterpret_cast<double2*>(buf + 2 * FIELD);     // [L][TYL][T]
  float2* __restrict__ mV = emit ? g.e0 : g.m0;
  float2* __restrict__ mE = emit ? g.e1 : g.m1;
  const size_t slab = (size_t)kx * NZ * y2 + ky;

  float2 w[E];
  load_twiddles<E>(w, g.twz, j);
  float2 A[E], Bf[E];                       // (D^ | V^), (J^z | -i kz V^)

  if constexpr (APPLY_J) {
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const size_t gi = slab + (size_t)(j + T * r) * y2;
      A[r] = g.m0[gi];
      Bf[r] = g.m1[gi];
    }
    fft_stage1<E, false>(A, w);
    fft_stage1<E, false>(Bf, w);
#pragma unroll
    for (int q = 0; q < E; ++q) {
      buf[q * QS + j * TYL + line] = A[q];
      buf[FIELD + q * QS + j * TYL + line] = Bf[q];
    }
    __syncthreads();
    fft_stage2<E, T, false>(A, j, [&](int q, int jj) { return buf[q * QS + jj * TYL + line]; });
    fft_stage2<E, T, false>(Bf, j, [&](int q, int jj) { return buf[FIELD + q * QS + jj * TYL + line]; });
  }

  // ---- per-mode update (a7), potential from charge (a2), pad-layer sums (a3, fp64) ------------------------
  double2 acc[kMaxLayers];
#pragma unroll
  for (int l = 0; l < kMaxLayers; ++l) acc[l] = make_double2(0.0, 0.0);
  const double kxd = g.kxd[kx], kyd = g.kyd[ky];
  const double kxy2 = kxd * kxd + kyd * kyd;
  const bool ret_x = (kx != nx / 2);
#pragma unroll
  for (int r = 0; r < E; ++r) {
    const int kz = j + T * r;
    const size_t gi = slab + (size_t)kz * y2;
    const bool ret = ret_x && (kz != NZ / 2);
    const double kzd = g.kzd[kz];
    double2 rr = g.rhat[gi];
    if constexpr (APPLY_J) {
      const float kzf = (float)kzd;
      rr.x -= (double)(A[r].x - kzf * Bf[r].y);
      rr.y -= (double)(A[r].y + kzf * Bf[r].x);
      if (!ret) rr = make_double2(0.0, 0.0);
      g.rhat[gi] = rr;
    }
    double2 src = rr;
    if constexpr (DELTA) {
      const double2 p = g.rhat_prev[gi];
      src.x -= p.x; src.y -= p.y;
      g.rhat_prev[gi] = rr;
    }
    const double k2 = kxy2 + kzd * kzd;
    const double gg = (ret && k2 > 0.0) ? gd.inv_n * fast_rcp(k2) : 0.0;
    const double2 v = make_double2(src.x * gg, src.y * gg);
    A[r] = make_float2((float)v.x, (float)v.y);
    Bf[r] = make_float2((float)(kzd * v.y), (float)(-kzd * v.x));   // -i kz V^
#pragma unroll
    for (int l = 0; l < kMaxLayers; ++l) {
      if (l < L) {
        double2 ww = g.twzd[(kz * g.layers[l]) & (NZ - 1)];
        ww.y = -ww.y;                                                 // e^{+i kz z_l}
        const double2 p = dmul(v, ww);
        acc[l].x += p.x; acc[l].y += p.y;
      }
    }
  }
  // ---- inverse z transforms ---------------------------------------------------------------------------
  fft_stage1<E, true>(A, w);
  fft_stage1<E, true>(Bf, w);
  if constexpr (APPLY_J) __syncthreads();            // the forward exchange has been read by everyone
#pragma unroll
  for (int q = 0; q < E; ++q) {
    buf[q * QS + j * TYL + line] = A[q];
    buf[FIELD + q * QS + j * TYL + line] = Bf[q];
  }
#pragma unroll
  for (int l = 0; l < kMaxLayers; ++l)
    if (l < L) red[(l * TYL + line) * T + j] = acc[l];
  __syncthreads();
  for (int i = tid; i < L * TYL; i += C::THREADS) {   // V~_rho(kx, z_l, ky) in fp64, fixed summation order
    double2 s = make_double2(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < T; ++k) { const double2 p = red[i * T + k]; s.x += p.x; s.y += p.y; }
    const int l = i / TYL, ln = i - l * TYL;
    (emit ? g.pl_e : g.pl)[((size_t)l * nx + kx) * y2 + ky0 + ln] = s;
  }
  fft_stage2<E, T, true>(A, j, [&](int q, int jj) { return buf[q * QS + jj * TYL + line]; });
  fft_stage2<E, T, true>(Bf, j, [&](int q, int jj) { return buf[FIELD + q * QS + jj * TYL + line]; });
#pragma unroll
  for (int r = 0; r < E; ++r) {
    const size_t gi = slab + (size_t)(j + T * r) * y2;
    mV[gi] = A[r];
    mE[gi] = Bf[r];
  }
}

}  // namespace wt
