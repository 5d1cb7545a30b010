// Size-generic kernels of wt_solve_H: any grid n = 2^a 3^b (mixed-radix Stockham passes in shared
// memory, fft.cuh).  The size-specialised kernels of solve_fast.cuh replace k_spectral and k_plane
// for the power-of-two sizes; both families read and write the same mixed-space arrays, so a plane
// kernel of one family can be combined with a z-line kernel of the other.
#pragma once
#include "fft.cuh"
#include "solve_common.cuh"

namespace wt {

// ------------------------------------------------------------------------------------------------
// k_spectral: z-line transforms + per-mode update.  grid (n_tiles, n_geoms), block 32*ty.
//   forward z DFT of D~, J~z;  r^ -= D^ + i kz J^z  (a7, fp64 state);  V^ = r^/|kappa|^2  (a2);
//   V~_rho at the pad layers in fp64 (a3);  inverse z DFT of V^ and -i kz V^  (a5, z part)
// ------------------------------------------------------------------------------------------------
// NZC, TYC: compile-time line length and lines per tile (0 = the run-time values): with them every index computation of the
// Stockham passes and of the tile loops folds to constants (configs[4]: nz = 384, 8 lines per tile).
template <bool APPLY_J, bool DELTA, int NZC, int TYC>
__device__ __forceinline__ void spectral_body(const GeomBatch& gb, const GridDev& gd, int emit) {
  const GeomDev& g = gb.g[blockIdx.y];
  const int nx = gd.nx, nz = NZC ? NZC : gd.nz, y2 = gd.y2, TY = TYC ? TYC : gd.ty;
  const int tiles = y2 / TY;
  const int kx = blockIdx.x / tiles, ky0 = (blockIdx.x % tiles) * TY;
  const int tid = threadIdx.x, bd = TYC ? 32 * TYC : blockDim.x;
  const int nelem = nz * TY;
  const int L = g.L;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* b0 = reinterpret_cast<float2*>(smraw);
  float2* b1 = b0 + nelem;
  float2* b2 = b1 + nelem;
  double2* red = reinterpret_cast<double2*>(b2 + nelem);   // [L][TY][32]
  // twiddles of the z transform: to shared memory while the predecessor runs (every butterfly of every pass
  // would otherwise fetch them from global memory in the middle of the kernel)
  float2* s_twz = reinterpret_cast<float2*>(red + (size_t)(L > 0 ? L : 1) * TY * 32);   // [nz]
  double2* s_twzd = reinterpret_cast<double2*>(s_twz + nz);                               // [nz] fp64 twiddles of the pad-layer sums
  double* s_kzd = reinterpret_cast<double*>(s_twzd + nz);                                 // [nz] z wavenumbers
  for (int i = tid; i < nz; i += bd) { s_twz[i] = g.twz[i]; s_twzd[i] = g.twzd[i]; s_kzd[i] = g.kzd[i]; }
  __syncthreads();
  pdl_wait();
  float2* mV = emit ? g.e0 : g.v0;
  float2* mE = emit ? g.e1 : g.v1;
  const size_t slab = (size_t)kx * nz * y2 + ky0;

  float2 *dres, *jres, *vb;
  if (APPLY_J) {
    for (int t = tid; t < nelem; t += bd) {
      const int z = t / TY, ty = t - z * TY;
      const size_t gi = slab + (size_t)z * y2 + ty;
      const float2 dx = g.m0[gi], dy = g.m1[gi];
      b0[t] = make_float2(dx.x + dy.x, dx.y + dy.y);   // D~ = i kx J~x + i ky J~y
      b2[t] = g.m2[gi];
    }
    __syncthreads();
    dres = fft_lines<float2>(b0, b1, nz, TY, 1, TY, s_twz, false);
    float2* free1 = (dres == b0) ? b1 : b0;
    jres = fft_lines<float2>(b2, free1, nz, TY, 1, TY, s_twz, false);
    vb = (jres == b2) ? free1 : b2;
  } else {
    vb = b0; dres = b1; jres = b2;
  }

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
    const double kzd = s_kzd[kz];
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
        double2 w = s_twzd[(kz * g.layers[l]) % nz];
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
  if (tid < L * TY) {                 // V~_rho(kx, z_l, ky) for this CTA's modes, fixed summation order
    double2 s = make_double2(0.0, 0.0);
    for (int i = 0; i < 32; ++i) { const double2 p = red[tid * 32 + i]; s.x += p.x; s.y += p.y; }
    const int l = tid / TY, j = tid - l * TY;
    (emit ? g.pl_e : g.pl)[((size_t)l * nx + kx) * y2 + ky0 + j] = s;
  }
  // inverse z transforms
  float2* vres = fft_lines<float2>(vb, jres, nz, TY, 1, TY, s_twz, true);
  float2* fr = (vres == vb) ? jres : vb;
  for (int t = tid; t < nelem; t += bd) {
    const int z = t / TY, tyy = t - z * TY;
    mV[slab + (size_t)z * y2 + tyy] = vres[t];
  }
  float2* eres = fft_lines<float2>(dres, fr, nz, TY, 1, TY, s_twz, true);
  for (int t = tid; t < nelem; t += bd) {
    const int z = t / TY, tyy = t - z * TY;
    mE[slab + (size_t)z * y2 + tyy] = eres[t];
  }
}

template <bool APPLY_J, bool DELTA>
__global__ void __launch_bounds__(256) k_spectral(const __grid_constant__ GeomBatch gb, GridDev gd, int substep, int emit) {
  pdl_trigger();
  if (substep >= gb.g[blockIdx.y].n_sub) { pdl_wait(); return; }
  if (gd.nz == 384 && gd.ty == 8) spectral_body<APPLY_J, DELTA, 384, 8>(gb, gd, emit);
  else spectral_body<APPLY_J, DELTA, 0, 0>(gb, gd, emit);
}

// ------------------------------------------------------------------------------------------------
// k_plane: xy-plane transforms.  grid (nz, n_geoms), block 256.
// Shared memory: two buffers of (nx/2)*(ny+1) float2 used either as a half-spectrum plane
// [kx][ky] (row stride y2) or as nx/2 complex lines of length ny, each packing the two real
// x-rows 2p (real part) and 2p+1 (imaginary part), line stride ny+1 (odd: conflict free).
//   V~ = V~_rho + sum_l Q^_l g~(z - z_l)  (a4);  E~ = -i kappa V~;  inverse xy DFT  (a5);
//   J = s dt_int E  (a6);  forward xy DFT;  out: i kx J~x, i ky J~y, J~z.   EMIT: H[n] = E/dt  (a8)
// ------------------------------------------------------------------------------------------------
template <bool EMIT>
__global__ void __launch_bounds__(256) k_plane(const __grid_constant__ GeomBatch gb, GridDev gd, int substep) {
  pdl_trigger();
  const GeomDev& g = gb.g[blockIdx.y];
  if (substep >= g.n_sub) { pdl_wait(); return; }
  const int nx = gd.nx, ny = gd.ny, nz = gd.nz, y2 = gd.y2;
  const int z = blockIdx.x;
  const int tid = threadIdx.x, bd = blockDim.x;
  const int nyp = ny + 1, hx = nx / 2;
  const int nspec = nx * y2, nline = hx * ny;
  const int bufsz = hx * nyp;
  extern __shared__ __align__(16) unsigned char smraw[];
  float2* w1 = reinterpret_cast<float2*>(smraw);
  float2* w2 = w1 + bufsz;
  // twiddles of the x and y transforms: to shared memory while the predecessor runs
  float2* s_twx = w2 + bufsz;                              // [nx]
  float2* s_twy = s_twx + nx;                              // [ny]
  for (int i = tid; i < nx; i += bd) s_twx[i] = g.twx[i];
  for (int i = tid; i < ny; i += bd) s_twy[i] = g.twy[i];
  __syncthreads();
  pdl_wait();
  const float2* mV = EMIT ? g.e0 : g.v0;
  const float2* mE = EMIT ? g.e1 : g.v1;
  const int L = g.L;
  const int slot = EMIT ? (*gd.step % kStageSlots) : 0;

  for (int comp = 0; comp < 3; ++comp) {
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
        const float kap = (comp == 0) ? g.kxf[kx] : g.kyf[ky];
        v = make_float2(kap * v.y, -kap * v.x);               // -i kappa V~
      }
      w1[t] = v;
    }
    __syncthreads();
    float2* r = fft_lines<float2>(w1, w2, nx, y2, 1, y2, s_twx, true);
    float2* o = (r == w1) ? w2 : w1;
    // pack two x-rows into one complex line with the Hermitian completion along y (Nyquist = 0)
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
    float2* e = fft_lines<float2>(o, r, ny, hx, nyp, 1, s_twy, true);
    float2* f = (e == o) ? r : o;
    if (EMIT) {
      // H[n] = E/dt into the staging slot, [slot][comp][z][x][y]
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
    float2* jf = fft_lines<float2>(e, f, ny, hx, nyp, 1, s_twy, false);
    float2* jo = (jf == e) ? f : e;
    for (int t = tid; t < hx * y2; t += bd) {
      const int p = t / y2, k = t - p * y2;
      const float2 zk = jf[p * nyp + k];
      const float2 zm = jf[p * nyp + (k == 0 ? 0 : ny - k)];
      jo[(2 * p) * y2 + k] = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
      jo[(2 * p + 1) * y2 + k] = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
    }
    __syncthreads();
    float2* jt = fft_lines<float2>(jo, jf, nx, y2, 1, y2, s_twx, false);
    for (int t = tid; t < nspec; t += bd) {
      const int kx = t / y2, ky = t - kx * y2;
      const float2 j = jt[t];
      const size_t gi = ((size_t)kx * nz + z) * y2 + ky;
      if (comp == 0) {
        const float kap = g.kxf[kx];
        g.m0[gi] = make_float2(-kap * j.y, kap * j.x);     // i kx J~x
      } else if (comp == 1) {
        const float kap = g.kyf[ky];
        g.m1[gi] = make_float2(-kap * j.y, kap * j.x);     // i ky J~y
      } else {
        g.m2[gi] = j;
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// k_transpose: staging -> H[((x*ny+y)*nz+z)*nt + t][comp] for the last cnt output steps, when the
// step counter n closes a group of kStageSlots steps (or is the last step); otherwise a no-op.
// YX = false: staging [slot][comp][z][x][y], grid (nz*nx, n_geoms);  YX = true: [slot][comp][z][y][x],
// grid (nz*ny, n_geoms).  block 256; dynamic smem kStageSlots*3*max(nx,ny) floats.
// ------------------------------------------------------------------------------------------------
template <bool YX>
__global__ void __launch_bounds__(256) k_transpose(const __grid_constant__ GeomBatch gb, GridDev gd) {
  pdl_trigger();
  pdl_wait();
  const int n = *gd.step;
  if (!((n + 1) % kStageSlots == 0 || n == gd.nt - 1)) return;
  const int cnt = n % kStageSlots + 1, t0 = n - cnt + 1;
  const GeomDev& g = gb.g[blockIdx.y];
  const int nx = gd.nx, ny = gd.ny, nz = gd.nz, nt = gd.nt;
  const int na = YX ? ny : nx;        // outer in-plane index (one per CTA)
  const int nb = YX ? nx : ny;        // inner in-plane index (contiguous in the staging)
  const int z = blockIdx.x / na, a = blockIdx.x - z * na;
  extern __shared__ float tile[];     // [cnt*3][nb]
  const int rows = cnt * 3;
  for (int t = threadIdx.x; t < rows * nb; t += blockDim.x) {
    const int j = t / nb, b = t - j * nb;          // j = slot*3 + comp
    tile[t] = g.stage[(((size_t)j * nz + z) * na + a) * nb + b];
  }
  __syncthreads();
  for (int t = threadIdx.x; t < rows * nb; t += blockDim.x) {
    const int b = t / rows, j = t - b * rows;
    const int x = YX ? b : a, y = YX ? a : b;
    g.H[((((size_t)x * ny + y) * nz + z) * nt + t0) * 3 + j] = tile[j * nb + b];
  }
}

__global__ void k_advance(int* step) {
  pdl_trigger();
  pdl_wait();
  *step += 1;
}

}  // namespace wt
