// Size-specialised kernels of wt_solve_H for power-of-two grids (the BASELINE configs 0-3):
// register-resident two-stage FFTs (regfft.cuh), all index arithmetic compile-time, one
// __syncthreads per shared-memory exchange.
//
//   k_plane_fast<N, E, EMIT>     one field component on one xy-plane of an N x N grid per CTA,
//                                N*N/(2E) threads;  grid (nz, 3 components, geometries)
//   k_pencil<NZ, E, TYL, ...>    z-lines of length NZ, one CTA per (kx, TYL consecutive ky), TYL*NZ/E threads
//
// Both read/write the mixed-space arrays [kx][z][ky] of solve_common.cuh exactly like the generic
// kernels (solve_generic.cuh), which remain the path for every other 2^a 3^b size.
#pragma once
#include "regfft.cuh"
#include "solve_common.cuh"

namespace wt {

template <int N> struct PlaneCfg {
  static constexpr int Y2 = N / 2;
  static constexpr int SX = N + 2;       // row stride of the transposed buffer [ky][x] (even: float4 reads)
  static constexpr int SU = N / 2 + 1;   // row stride of the unpack buffer [k][p2] (odd: strided reads conflict free)
  static constexpr int BUF = (Y2 * SX > N * SU) ? Y2 * SX : N * SU;   // float2 per buffer (>= N*Y2)
};

// ------------------------------------------------------------------------------------------------
// k_plane_fast.  grid (nz, 3, n_geoms), block N*N/(2E), dynamic smem 2 * BUF * 8 bytes.
//   V~ = V~_rho + sum_l Q^_l g~(z - z_l)  (a4);  E~_c = -i kappa_c V~;  inverse xy DFT  (a5);
//   J_c = s dt_int E_c  (a6);  forward xy DFT;  out_c = i kappa_c J~_c (c = x, y) or J~_z.
//   EMIT: H_c[n] = E_c/dt into the staging slot  (a8)
//
// x-phases: thread (ky = tid % Y2, j = tid / Y2) holds kx (or x) = j + T r, r < E, of line ky.
// y-phases: thread (p2 = tid % Y2, j) holds k (or y) = j + T r of the complex line p2 that packs the
//           real x-rows 2 p2 (real part) and 2 p2 + 1 (imaginary part).
// Exchanges ping-pong between two buffers P and Q: six barriers per plane.
// ------------------------------------------------------------------------------------------------
template <int N, int E, bool EMIT>
__global__ void __launch_bounds__(N * N / (2 * E), (N <= 64) ? 3 : (N == 96 ? 2 : 1))   // 80 registers, no spills (4 CTAs/SM at 64 registers spilled and measured 1 us slower per substep)
k_plane_fast(const __grid_constant__ GeomBatch gb, GridDev gd, int substep) {
  using C = PlaneCfg<N>;
  constexpr int Y2 = C::Y2, T = N / E, SX = C::SX, SU = C::SU, BUF = C::BUF;
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.z];
  if (substep >= g.n_sub) { pdl_wait(); return; }
  const int nz = gd.nz, z = blockIdx.x, comp = blockIdx.y;
  const int tid = threadIdx.x;
  const int ln = tid % Y2;     // line within the phase: ky (x-phases) or p2 (y-phases)
  const int j = tid / Y2;      // position of the thread within its line
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* P = reinterpret_cast<float2*>(smraw);
  float2* Q = P + BUF;
  const int L = g.L;

  // per-thread twiddles W_N^{jq}: registers for E <= 16; a [T][E] table in shared memory for E = 24 (N = 96), where 48 more
  // registers would leave one CTA per SM
  constexpr bool TW_SMEM = E > 16;
  __shared__ float2 s_w[TW_SMEM ? T * E : 1];
  float2 w_reg[TW_SMEM ? 1 : E];
  const float2* w_tab = s_w + (TW_SMEM ? j * E : 0);
  if constexpr (TW_SMEM) {
    for (int i = tid; i < T * E; i += N * N / (2 * E)) s_w[i] = __ldg(g.twx + (i / E) * (i % E));   // N x N plane: twx == twy
  } else {
    load_twiddles<E>(w_reg, g.twx, j);
  }
  // small tables that are needed in the middle and at the end of the kernel go to shared memory now, while the
  // predecessor is still running: a global load there would stall every warp of the CTA with nothing to overlap
  __shared__ float s_sdt[256];
  __shared__ float s_kx[N];
  if (!EMIT)
    for (int i = tid; i < 256; i += N * N / (2 * E)) s_sdt[i] = __ldg(g.sdt + i);
  for (int i = tid; i < N; i += N * N / (2 * E)) s_kx[i] = __ldg(g.kxf + i);

  // conductivity ids of this thread's nodes in the y-phases: rows 2 ln, 2 ln + 1 at y = j + T r
  unsigned short sid[E];
  if (!EMIT) {
    const unsigned short* st = reinterpret_cast<const unsigned short*>(g.sig_t + (size_t)z * N * N);
#pragma unroll
    for (int r = 0; r < E; ++r) sid[r] = __ldg(st + ((j + T * r) * N + 2 * ln) / 2);
  }

  const float kyv = __ldg(g.kyf + ln);
  __syncthreads();
  pdl_wait();
  float2 X[E];
  // ---- load: V~ = V~_rho + sum_l Q^_l g~(z - z_l) (the boundary source, a4); E~ = -i kappa V~ ------------
  {
    const float2* __restrict__ src = EMIT ? (comp == 2 ? g.e1 : g.e0) : (comp == 2 ? g.v1 : g.v0);
    const float* __restrict__ tab = (comp == 2) ? g.gzt : g.gt;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int kx = j + T * r;
      X[r] = src[((size_t)kx * nz + z) * Y2 + ln];
    }
    for (int l = 0; l < L; ++l) {
      int dz = z - g.layers[l];
      dz = dz < 0 ? dz + nz : dz;
      const float2* __restrict__ qh = g.qh + (size_t)l * N * Y2 + ln;
      const float* __restrict__ tl = tab + (size_t)dz * Y2 + ln;
#pragma unroll
      for (int r = 0; r < E; ++r) {
        const int kx = j + T * r;
        const float2 qv = qh[kx * Y2];
        const float gv = __ldg(tl + (size_t)kx * nz * Y2);
        X[r].x += qv.x * gv; X[r].y += qv.y * gv;
      }
    }
    if (comp < 2) {
#pragma unroll
      for (int r = 0; r < E; ++r) {
        const float kap = (comp == 0) ? s_kx[j + T * r] : kyv;
        X[r] = make_float2(kap * X[r].y, -kap * X[r].x);       // -i kappa V~
      }
    }
  }
  // ---- A: inverse transform along x ---------------------------------------------------------------------
  if constexpr (TW_SMEM) fft_stage1<E, true>(X, w_tab); else fft_stage1<E, true>(X, w_reg);
#pragma unroll
  for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[q];
  __syncthreads();
  fft_stage2<E, T, true>(X, j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
  // ---- transpose: [ky][x] so that a y-phase thread reads the row pair (2 p2, 2 p2 + 1) as one float4 -------
#pragma unroll
  for (int r = 0; r < E; ++r) Q[ln * SX + j + T * r] = X[r];
  __syncthreads();
  // Hermitian completion along y of the two packed real rows (Nyquist = 0): z[k] = a[k] + i b[k]
#pragma unroll
  for (int r = 0; r < E; ++r) {
    if (r < E / 2) {                               // k = j + T r < Y2
      const float4 ab = *reinterpret_cast<const float4*>(&Q[(j + T * r) * SX + 2 * ln]);
      X[r] = make_float2(ab.x - ab.w, ab.y + ab.z);
    } else {                                       // k >= Y2: mirror k' = N - k in [1, Y2]
      const int km = N - (j + T * r);
      if (km == Y2) {
        X[r] = make_float2(0.f, 0.f);
      } else {
        const float4 ab = *reinterpret_cast<const float4*>(&Q[km * SX + 2 * ln]);
        X[r] = make_float2(ab.x + ab.w, ab.z - ab.y);
      }
    }
  }
  // ---- B: inverse transform along y -> E at the nodes (rows 2 ln | 2 ln + 1, y = j + T r) -----------------
  if constexpr (TW_SMEM) fft_stage1<E, true>(X, w_tab); else fft_stage1<E, true>(X, w_reg);
#pragma unroll
  for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[q];
  __syncthreads();
  fft_stage2<E, T, true>(X, j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
  if constexpr (EMIT) {
    // (a8) H[n] = E/dt into the staging slot [slot][comp][z][y][x]
    const int slot = *gd.step % kStageSlots;
    float2* st = reinterpret_cast<float2*>(g.stage + (((size_t)slot * 3 + comp) * nz + z) * (size_t)(N * N));
#pragma unroll
    for (int r = 0; r < E; ++r) st[((j + T * r) * N + 2 * ln) / 2] = make_float2(X[r].x * g.inv_dt, X[r].y * g.inv_dt);
    return;
  }
  // ---- conduction current J = (s dt_int) E, nodewise (a6, R17) ----------------------------------------------
#pragma unroll
  for (int r = 0; r < E; ++r) {
    X[r].x *= s_sdt[sid[r] & 0xff];
    X[r].y *= s_sdt[sid[r] >> 8];
  }
  // ---- C: forward transform along y ---------------------------------------------------------------------
  if constexpr (TW_SMEM) fft_stage1<E, false>(X, w_tab); else fft_stage1<E, false>(X, w_reg);
#pragma unroll
  for (int q = 0; q < E; ++q) Q[(q * T + j) * Y2 + ln] = X[q];
  __syncthreads();
  fft_stage2<E, T, false>(X, j, [&](int q, int jj) { return Q[(q * T + jj) * Y2 + ln]; });
  // ---- unpack the two real rows' half spectra: [k][p2], read back with ln = ky ------------------------------
#pragma unroll
  for (int r = 0; r < E; ++r) P[(j + T * r) * SU + ln] = X[r];
  __syncthreads();
  {
    const int km = (N - ln) % N;
    const bool odd = j & 1;                          // x = j + T r, T even
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int p2 = (j + T * r) >> 1;
      const float2 zk = P[ln * SU + p2], zm = P[km * SU + p2];
      X[r] = odd ? make_float2(0.5f * (zk.y + zm.y), 0.5f * (zm.x - zk.x))
                 : make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
    }
  }
  // ---- D: forward transform along x ---------------------------------------------------------------------
  if constexpr (TW_SMEM) fft_stage1<E, false>(X, w_tab); else fft_stage1<E, false>(X, w_reg);
#pragma unroll
  for (int q = 0; q < E; ++q) Q[(q * T + j) * Y2 + ln] = X[q];
  __syncthreads();
  fft_stage2<E, T, false>(X, j, [&](int q, int jj) { return Q[(q * T + jj) * Y2 + ln]; });
  // ---- out: i kx J~x | i ky J~y | J~z ----------------------------------------------------------------------
  {
    float2* __restrict__ dst = (comp == 0) ? g.m0 : (comp == 1) ? g.m1 : g.m2;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int kx = j + T * r;
      float2 o = X[r];
      if (comp < 2) {
        const float kap = (comp == 0) ? s_kx[kx] : kyv;
        o = make_float2(-kap * o.y, kap * o.x);
      }
      dst[((size_t)kx * nz + z) * Y2 + ln] = o;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// k_pencil: z-line transforms + per-mode update (a7, a2), pad-layer potentials in fp64 (a3),
// inverse z transforms (a5, z part).  grid (nx * y2/TYL, n_geoms), block TYL * NZ/E.
// Thread (line = tid % TYL, j = tid / TYL) holds z (or kz) = j + T r, r < E, of line ky0 + line.
// dynamic smem: 2 fields * E * QS float2 + LT * TYL * T double2.  LT = compile-time bound on the
// number of pad layers (2 or kMaxLayers).
// ------------------------------------------------------------------------------------------------
template <int NZ, int E, int TYL> struct PencilCfg {
  static constexpr int T = NZ / E;
  static constexpr int PAD = (TYL < 16) ? 16 - TYL : 0;   // skews consecutive q rows across the banks
  static constexpr int QS = T * TYL + PAD;                // float2 per q row of an exchange buffer
  static constexpr int FIELD = E * QS;
  static constexpr int THREADS = T * TYL;
};

// reciprocal of a positive, normal double by Newton iteration from the fp32 estimate (rel. error ~1e-16)
__device__ __forceinline__ double fast_rcp(double a) {
  float xf;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(xf) : "f"((float)a));
  double x = (double)xf;
  x = x * (2.0 - a * x);
  x = x * (2.0 - a * x);
  return x;
}

template <int NZ, int E, int TYL, int LT, bool APPLY_J, bool DELTA>
__global__ void __launch_bounds__(PencilCfg<NZ, E, TYL>::THREADS)
k_pencil(const __grid_constant__ GeomBatch gb, GridDev gd, int substep, int emit) {
  using C = PencilCfg<NZ, E, TYL>;
  constexpr int T = C::T, QS = C::QS, FIELD = C::FIELD;
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.y];
  if (substep >= g.n_sub) { pdl_wait(); return; }
  const int nx = gd.nx, y2 = gd.y2;
  const int tiles = y2 / TYL;
  const int kx = blockIdx.x / tiles, ky0 = (blockIdx.x % tiles) * TYL;
  const int tid = threadIdx.x;
  const int line = tid % TYL, j = tid / TYL;
  const int ky = ky0 + line;
  const int L = g.L;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* buf = reinterpret_cast<float2*>(smraw);                 // [2][E][QS]
  double2* red = reinterpret_cast<double2*>(buf + 2 * FIELD);     // [LT][TYL][T]
  const size_t slab = (size_t)kx * NZ * y2 + ky;

  float2 w[E];
  load_twiddles<E>(w, g.twz, j);
  float2 A[E], Bf[E];                       // (D^ | V^), (J^z | -i kz V^)
  pdl_wait();

  if constexpr (APPLY_J) {
    const float2* __restrict__ m0 = g.m0 + slab;
    const float2* __restrict__ m1 = g.m1 + slab;
    const float2* __restrict__ m2 = g.m2 + slab;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const size_t o = (size_t)(j + T * r) * y2;
      const float2 a = m0[o], b = m1[o];
      A[r] = make_float2(a.x + b.x, a.y + b.y);      // D~ = i kx J~x + i ky J~y
      Bf[r] = m2[o];
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
  double2 acc[LT];
#pragma unroll
  for (int l = 0; l < LT; ++l) acc[l] = make_double2(0.0, 0.0);
  const double kxd = g.kxd[kx], kyd = g.kyd[ky];
  const double kxy2 = kxd * kxd + kyd * kyd;
  const bool ret_x = (kx != nx / 2);
  double2* __restrict__ rh = g.rhat + slab;
  double2* __restrict__ rp = g.rhat_prev + slab;
#pragma unroll
  for (int r = 0; r < E; ++r) {
    const int kz = j + T * r;
    const size_t o = (size_t)kz * y2;
    const bool ret = ret_x && (kz != NZ / 2);
    const double kzd = g.kzd[kz];
    double2 rr = rh[o];
    if constexpr (APPLY_J) {
      const float kzf = (float)kzd;
      rr.x -= (double)(A[r].x - kzf * Bf[r].y);
      rr.y -= (double)(A[r].y + kzf * Bf[r].x);
      if (!ret) rr = make_double2(0.0, 0.0);
      rh[o] = rr;
    }
    double2 src = rr;
    if constexpr (DELTA) {
      const double2 p = rp[o];
      src.x -= p.x; src.y -= p.y;
      rp[o] = rr;
    }
    const double k2 = kxy2 + kzd * kzd;
    const double gg = (ret && k2 > 0.0) ? gd.inv_n * fast_rcp(k2) : 0.0;
    const double2 v = make_double2(src.x * gg, src.y * gg);
    A[r] = make_float2((float)v.x, (float)v.y);
    Bf[r] = make_float2((float)(kzd * v.y), (float)(-kzd * v.x));   // -i kz V^
#pragma unroll
    for (int l = 0; l < LT; ++l) {
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
  for (int l = 0; l < LT; ++l)
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
  {
    float2* __restrict__ oV = (emit ? g.e0 : g.v0) + slab;
    float2* __restrict__ oE = (emit ? g.e1 : g.v1) + slab;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const size_t o = (size_t)(j + T * r) * y2;
      oV[o] = A[r];
      oE[o] = Bf[r];
    }
  }
}


// ------------------------------------------------------------------------------------------------
// k_pencil2: the z-line kernel with ONE field per thread (twice the threads of k_pencil, half the
// registers): threads (f = 0, line, j) transform D~ / V^, threads (f = 1, line, j) transform
// J~z / -i kz V^.  The per-mode update needs both fields of a mode: after the forward transform the
// spectra pass through a kz-indexed shared buffer, each thread updates E/2 modes of its line
// in place (V^ and -i kz V^ overwrite D^ and J^z), and the inverse transforms read them back.
// grid (nx * y2/TYL, n_geoms), block 2 * TYL * NZ/E.
// dynamic smem: 2 fields * E * QS float2 (exchange) + 2 * NZ * TYL float2 (kz-indexed) + LT * TYL * 2T double2.
// ------------------------------------------------------------------------------------------------
template <int NZ, int E, int TYL, int LT, bool APPLY_J, bool DELTA>
__global__ void __launch_bounds__(2 * PencilCfg<NZ, E, TYL>::THREADS, 2)
k_pencil2(const __grid_constant__ GeomBatch gb, GridDev gd, int substep, int emit) {
  using C = PencilCfg<NZ, E, TYL>;
  constexpr int T = C::T, QS = C::QS, FIELD = C::FIELD, HT = C::THREADS;   // HT threads per field
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.y];
  if (substep >= g.n_sub) { pdl_wait(); return; }
  const int nx = gd.nx, y2 = gd.y2;
  const int tiles = y2 / TYL;
  const int kx = blockIdx.x / tiles, ky0 = (blockIdx.x % tiles) * TYL;
  const int tid = threadIdx.x;
  const int f = tid / HT, th = tid % HT;
  const int line = th % TYL, j = th / TYL;
  const int ky = ky0 + line;
  const int L = g.L;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* buf = reinterpret_cast<float2*>(smraw) + f * FIELD;                  // [2][E][QS]   exchange of this field
  float2* kzb = reinterpret_cast<float2*>(smraw) + 2 * FIELD;                  // [2][NZ][TYL] kz-indexed spectra
  double2* red = reinterpret_cast<double2*>(kzb + 2 * NZ * TYL);               // [LT][TYL][2T]
  const size_t slab = (size_t)kx * NZ * y2 + ky;

  float2 w[E];
  load_twiddles<E>(w, g.twz, j);
  float2 X[E];
  // wavenumbers and fp64 twiddles of the per-mode update: to shared memory during the prologue (a global
  // load in the middle of the kernel stalls all warps of the CTA with nothing to overlap)
  __shared__ double s_kz[NZ];
  __shared__ double2 s_twz[NZ];
  for (int i = tid; i < NZ; i += 2 * HT) { s_kz[i] = g.kzd[i]; s_twz[i] = g.twzd[i]; }
  const double kxd = g.kxd[kx], kyd = g.kyd[ky];
  __syncthreads();
  pdl_wait();

  if constexpr (APPLY_J) {
    if (f == 0) {
      const float2* __restrict__ m0 = g.m0 + slab;
      const float2* __restrict__ m1 = g.m1 + slab;
#pragma unroll
      for (int r = 0; r < E; ++r) {
        const size_t o = (size_t)(j + T * r) * y2;
        const float2 a = m0[o], b = m1[o];
        X[r] = make_float2(a.x + b.x, a.y + b.y);      // D~ = i kx J~x + i ky J~y
      }
    } else {
      const float2* __restrict__ m2 = g.m2 + slab;
#pragma unroll
      for (int r = 0; r < E; ++r) X[r] = m2[(size_t)(j + T * r) * y2];
    }
    fft_stage1<E, false>(X, w);
#pragma unroll
    for (int q = 0; q < E; ++q) buf[q * QS + j * TYL + line] = X[q];
    __syncthreads();
    fft_stage2<E, T, false>(X, j, [&](int q, int jj) { return buf[q * QS + jj * TYL + line]; });
    // X[p] = spectrum at kz = j + T p: into the kz-indexed buffer
#pragma unroll
    for (int p = 0; p < E; ++p) kzb[(f * NZ + j + T * p) * TYL + line] = X[p];
    __syncthreads();
  }

  // ---- per-mode update (a7), potential from charge (a2), pad-layer sums (a3, fp64) ------------------------
  // thread (f, line, j) owns the modes kz = j + T (2 i + f), i < E/2
  {
    double2 acc[LT];
#pragma unroll
    for (int l = 0; l < LT; ++l) acc[l] = make_double2(0.0, 0.0);
    const double kxy2 = kxd * kxd + kyd * kyd;
    const bool ret_x = (kx != nx / 2);
    double2* __restrict__ rh = g.rhat + slab;
    double2* __restrict__ rp = g.rhat_prev + slab;
#pragma unroll
    for (int i = 0; i < E / 2; ++i) {
      const int kz = j + T * (2 * i + f);
      const size_t o = (size_t)kz * y2;
      const bool ret = ret_x && (kz != NZ / 2);
      const double kzd = s_kz[kz];
      double2 rr = rh[o];
      if constexpr (APPLY_J) {
        const float2 D = kzb[kz * TYL + line], J = kzb[(NZ + kz) * TYL + line];
        const float kzf = (float)kzd;
        rr.x -= (double)(D.x - kzf * J.y);
        rr.y -= (double)(D.y + kzf * J.x);
        if (!ret) rr = make_double2(0.0, 0.0);
        rh[o] = rr;
      }
      double2 src = rr;
      if constexpr (DELTA) {
        const double2 p = rp[o];
        src.x -= p.x; src.y -= p.y;
        rp[o] = rr;
      }
      const double k2 = kxy2 + kzd * kzd;
      const double gg = (ret && k2 > 0.0) ? gd.inv_n * fast_rcp(k2) : 0.0;
      const double2 v = make_double2(src.x * gg, src.y * gg);
      kzb[kz * TYL + line] = make_float2((float)v.x, (float)v.y);
      kzb[(NZ + kz) * TYL + line] = make_float2((float)(kzd * v.y), (float)(-kzd * v.x));   // -i kz V^
#pragma unroll
      for (int l = 0; l < LT; ++l) {
        if (l < L) {
          double2 ww = s_twz[(kz * g.layers[l]) & (NZ - 1)];
          ww.y = -ww.y;                                                 // e^{+i kz z_l}
          const double2 p = dmul(v, ww);
          acc[l].x += p.x; acc[l].y += p.y;
        }
      }
    }
#pragma unroll
    for (int l = 0; l < LT; ++l)
      if (l < L) red[(l * TYL + line) * (2 * T) + f * T + j] = acc[l];
  }
  __syncthreads();
  for (int i = tid; i < L * TYL; i += 2 * HT) {       // V~_rho(kx, z_l, ky) in fp64, fixed summation order
    double2 s = make_double2(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < 2 * T; ++k) { const double2 p = red[i * (2 * T) + k]; s.x += p.x; s.y += p.y; }
    const int l = i / TYL, ln = i - l * TYL;
    (emit ? g.pl_e : g.pl)[((size_t)l * nx + kx) * y2 + ky0 + ln] = s;
  }
  // ---- inverse z transform of this thread's field --------------------------------------------------------
#pragma unroll
  for (int r = 0; r < E; ++r) X[r] = kzb[(f * NZ + j + T * r) * TYL + line];
  fft_stage1<E, true>(X, w);
#pragma unroll
  for (int q = 0; q < E; ++q) buf[q * QS + j * TYL + line] = X[q];
  __syncthreads();
  fft_stage2<E, T, true>(X, j, [&](int q, int jj) { return buf[q * QS + jj * TYL + line]; });
  {
    float2* __restrict__ out = (f == 0 ? (emit ? g.e0 : g.v0) : (emit ? g.e1 : g.v1)) + slab;
#pragma unroll
    for (int r = 0; r < E; ++r) out[(size_t)(j + T * r) * y2] = X[r];
  }
}

}  // namespace wt
