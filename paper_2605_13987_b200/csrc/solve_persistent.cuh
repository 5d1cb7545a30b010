// Persistent solver of wt_solve_H: ONE cooperative launch per output step of H (n_sub Euler substeps +
// the emit of H[n]) for one geometry, one CTA per SM, phases separated by grid barriers instead of
// kernel boundaries (the per-substep kernel chain of solve_chain.cu pays a launch, a first-load round trip
// and a store drain three times per substep: profiles/r1_solve.md).
//
// Method as in solve.cu (Fig. 3 :109; R1-R20).  One Euler substep =
//   plane phase   all CTAs: (z, component) units, E~ = -i kappa V~ (a5), inverse xy DFT, J = s dt_int E (a6),
//                 forward xy DFT, i kx J~x, i ky J~y, J~z                                           -> m0, m1, m2
//   -- grid barrier --
//   z-line phase  Z CTAs own fixed tiles of z-lines (kx, TYL ky):
//      pass A     forward z DFT; r^ -= D^ + i kz J^z (a7, fp64 state); V^_rho = r^/|kappa|^2 (a2); potentials of
//                 the pad layers (fp64) and from them this CTA's contribution to V_rho at EVERY pad node (a3),
//                 added to a global int64 fixed-point accumulator per pad (integer adds commute: deterministic)
//      boundary   B CTAs (the SMs the z-lines leave idle): rhs = V_pad - V_rho|_B;
//                 Q' = Ainv rhs: "adjusted, in magnitude, to enforce the boundary conditions"
//      pass B     spectrum of the boundary point charges for the CTA's own lines; V^ = V^_rho + Q^/|kappa|^2, i.e. the
//                 translated fundamental solutions of PAPER.md:97 summed in spectral space (a4);
//                 inverse z DFT of V^ and -i kz V^                                                  -> v0, v1
//      With one tile per z-line group (BASELINE configs 0, 1, 3) the fp64 state of the tile lives in shared memory and
//      its 1/|kappa|^2 factors in registers for the whole launch, and V^_rho waits in shared memory for the charges
//      (RES); otherwise (config 2) the state stays in global memory and pass B forms V^ from it again.
//   -- grid barrier --
// and every n_sub substeps the same phases run on the increment r^ - r^_prev with the pads at 0 V and write
// H[n] = E/dt (a8) into the staging buffer, which a last phase transposes into the time-innermost table.
// Spins (grid barrier, boundary hand-over) are bounded: on a time-out the kernel sets ctl->abort, every CTA
// leaves, later launches return at once and k_persist_finish poisons the table with NaN -- a wrong launch
// configuration can cost a second, never a hang.
#pragma once
#include <type_traits>

#include "solve_fast.cuh"

namespace wt {

struct PersistCtl {                 // device control block, zeroed before the first launch of a solve
  unsigned long long bar;           // grid-barrier arrivals (monotonic)
  unsigned long long cnt_part;      // Z CTAs that have published their pad contributions (monotonic)
  unsigned long long cnt_rhs;       // B CTAs that have published their slice of rhs
  unsigned long long cnt_q;         // B CTAs that have published their slice of Q'
  int abort;
};

struct PersistArgs {
  GeomDev g;
  GridDev gd;
  PersistCtl* ctl;
  long long* fix;                   // [2][Bs]: V_rho at the pads as int64 fixed point (2^42), double buffered by episode parity
  const int* pad_x;                 // [B] group order
  const int* pad_l;                 // [B] layer index of the pad
  int lpoff[kMaxLayers + 1];        // pads of layer l = [lpoff[l], lpoff[l+1])
  int n_z_cta, n_b_cta;
  int ainv_in_smem;                 // the B CTA's rows of Ainv live in shared memory for the whole launch
  unsigned smem_persist_off;        // byte offset of the persistent region in the dynamic shared memory
  int step;                         // index n of the output step this launch produces
  int n_sub;                        // Euler substeps before the emit (0 for n = 0)
  unsigned long long bar0, epi0;    // grid barriers / boundary episodes completed by earlier launches
#ifdef WTIDE_DEBUG
  unsigned long long* stamps;       // [n_cta][64] globaltimer stamps of thread 0 during output step 2 (timing experiments)
#endif
};

constexpr long long kSpinLimit = 4000000000LL;     // cycles (about two seconds)
constexpr int kPersistThreads = 512;

__device__ __forceinline__ void group_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
// thread 0 of a CTA: wait until *ctr >= target; false on time-out / abort
__device__ __forceinline__ bool spin_until(const unsigned long long* ctr, unsigned long long target, int* abort_flag) {
  const long long t0 = clock64();
  unsigned it = 0;
  while (ld_acquire_u64(ctr) < target) {
    if ((++it & 63u) == 0) {
      if (*reinterpret_cast<volatile int*>(abort_flag)) return false;
      if (clock64() - t0 > kSpinLimit) { atomicExch(abort_flag, 1); return false; }
    }
  }
  return true;
}
// publish: everything this CTA wrote before is visible to whoever observes the increment
__device__ __forceinline__ void cta_signal(unsigned long long* ctr) {
  __syncthreads();
  if (threadIdx.x == 0) { __threadfence(); atomicAdd(ctr, 1ULL); }
}
__device__ __forceinline__ bool cta_wait(const unsigned long long* ctr, unsigned long long target, int* abort_flag, int* s_ok) {
  if (threadIdx.x == 0) *s_ok = spin_until(ctr, target, abort_flag) ? 1 : 0;
  __syncthreads();
  const bool ok = *s_ok != 0;
  __syncthreads();
  return ok;
}

#ifdef WTIDE_DEBUG
// fine stamps of thread 0 (group 0) inside the z passes: slots 32.. of the CTA's row, substep 1 of output step 2 only
__shared__ int g_fine_on;
#define FSTAMP(k) do { if (a.stamps && a.step == 2 && threadIdx.x == 0 && g_fine_on) { unsigned long long t_; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_)); a.stamps[(size_t)blockIdx.x * 64 + 32 + (k)] = t_; } } while (0)
#else
#define FSTAMP(k) do { } while (0)
#endif
__device__ __forceinline__ float2 ldcg2(const float2* p) { return __ldcg(p); }
__device__ __forceinline__ double2 dmulc(double2 a, double2 w) {      // a * conj(w)
  return make_double2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y);
}

// ------------------------------------------------------------------------------------------------
// plane_unit<N, E, EMIT, NC>: the xy-plane transforms of k_plane_fast (solve_fast.cuh) for a GROUP of N*N/(2E)
// threads of the CTA, without the boundary source (the z-line phase has already added it).
//   NC = 2  components x and y of plane z together: V~ is read once, the two transforms run interleaved (one barrier per
//           exchange for both), and D~ = i kx J~x + i ky J~y leaves as ONE array (m0)
//   NC = 1  component z: E~z -> J~z (m2)
// Buffers: P[c], Q[c] (c < NC) of PlaneCfg<N>::BUF float2 each, at P0 + (2 c) BUF and P0 + (2 c + 1) BUF.
// ------------------------------------------------------------------------------------------------
template <int N, int E>
__device__ __forceinline__ void plane_load(float2 (&V)[E], const float2* __restrict__ src, int nz, int z, int tid) {
  constexpr int Y2 = N / 2, T = N / E;
  const int ln = tid % Y2, j = tid / Y2;
#pragma unroll
  for (int r = 0; r < E; ++r) V[r] = ldcg2(src + ((size_t)(j + T * r) * nz + z) * Y2 + ln);
}

template <int N, int E, bool EMIT, int NC>
__device__ __forceinline__ void plane_unit(const GeomDev& g, int nz, int z, int comp1, const float2 (&V)[E], float2* P0,
                                           const float* s_sdt, const float* s_kx, int tid, int bar_id, int slot) {
  using C = PlaneCfg<N>;
  constexpr int Y2 = C::Y2, T = N / E, SX = C::SX, SU = C::SU, NT = N * N / (2 * E), BUF = C::BUF;
  const int ln = tid % Y2, j = tid / Y2;
  float2 w[E];
  load_twiddles<E>(w, g.twx, j);
  unsigned short sid[E];
  if (!EMIT) {
    const unsigned short* st = reinterpret_cast<const unsigned short*>(g.sig_t + (size_t)z * N * N);
#pragma unroll
    for (int r = 0; r < E; ++r) sid[r] = __ldg(st + ((j + T * r) * N + 2 * ln) / 2);
  }
  const float kyv = __ldg(g.kyf + ln);
  float2 X[NC][E];
#pragma unroll
  for (int r = 0; r < E; ++r) {
    const float2 v = V[r];
    if constexpr (NC == 2) {
      const float kx = s_kx[j + T * r];
      X[0][r] = make_float2(kx * v.y, -kx * v.x);        // -i kx V~
      X[1][r] = make_float2(kyv * v.y, -kyv * v.x);      // -i ky V~
    } else {
      if (comp1 == 2) {
        X[0][r] = v;                                     // E~z
      } else {
        const float kap = (comp1 == 0) ? s_kx[j + T * r] : kyv;
        X[0][r] = make_float2(kap * v.y, -kap * v.x);    // -i kappa V~
      }
    }
  }
  // ---- A: inverse transform along x
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + (2 * c) * BUF;
    fft_stage1<E, true>(X[c], w);
#pragma unroll
    for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + (2 * c) * BUF;
    float2* Q = P + BUF;
    fft_stage2<E, T, true>(X[c], j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
#pragma unroll
    for (int r = 0; r < E; ++r) Q[ln * SX + j + T * r] = X[c][r];
  }
  group_sync(bar_id, NT);
  // Hermitian completion along y of the two packed real rows (Nyquist = 0); B: inverse transform along y
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + (2 * c) * BUF;
    float2* Q = P + BUF;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      if (r < E / 2) {
        const float4 ab = *reinterpret_cast<const float4*>(&Q[(j + T * r) * SX + 2 * ln]);
        X[c][r] = make_float2(ab.x - ab.w, ab.y + ab.z);
      } else {
        const int km = N - (j + T * r);
        if (km == Y2) {
          X[c][r] = make_float2(0.f, 0.f);
        } else {
          const float4 ab = *reinterpret_cast<const float4*>(&Q[km * SX + 2 * ln]);
          X[c][r] = make_float2(ab.x + ab.w, ab.z - ab.y);
        }
      }
    }
    fft_stage1<E, true>(X[c], w);
#pragma unroll
    for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + (2 * c) * BUF;
    fft_stage2<E, T, true>(X[c], j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
  }
  if constexpr (EMIT) {
    // (a8) H[n] = E/dt into the staging slot [slot][comp][z][y][x]
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      const int comp = (NC == 2) ? c : comp1;
      float2* st = reinterpret_cast<float2*>(g.stage + (((size_t)slot * 3 + comp) * nz + z) * (size_t)(N * N));
#pragma unroll
      for (int r = 0; r < E; ++r) st[((j + T * r) * N + 2 * ln) / 2] = make_float2(X[c][r].x * g.inv_dt, X[c][r].y * g.inv_dt);
    }
    group_sync(bar_id, NT);                     // P is rewritten by the group's next unit
    return;
  }
  // ---- J = (s dt_int) E nodewise (a6); C: forward transform along y
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* Q = P0 + (2 * c + 1) * BUF;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      X[c][r].x *= s_sdt[sid[r] & 0xff];
      X[c][r].y *= s_sdt[sid[r] >> 8];
    }
    fft_stage1<E, false>(X[c], w);
#pragma unroll
    for (int q = 0; q < E; ++q) Q[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + (2 * c) * BUF;
    float2* Q = P + BUF;
    fft_stage2<E, T, false>(X[c], j, [&](int q, int jj) { return Q[(q * T + jj) * Y2 + ln]; });
#pragma unroll
    for (int r = 0; r < E; ++r) P[(j + T * r) * SU + ln] = X[c][r];
  }
  group_sync(bar_id, NT);
  // unpack the two real rows' half spectra; D: forward transform along x
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + (2 * c) * BUF;
    float2* Q = P + BUF;
    const int km = (N - ln) % N;
    const bool odd = j & 1;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int p2 = (j + T * r) >> 1;
      const float2 zk = P[ln * SU + p2], zm = P[km * SU + p2];
      X[c][r] = odd ? make_float2(0.5f * (zk.y + zm.y), 0.5f * (zm.x - zk.x))
                    : make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
    }
    fft_stage1<E, false>(X[c], w);
#pragma unroll
    for (int q = 0; q < E; ++q) Q[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* Q = P0 + (2 * c + 1) * BUF;
    fft_stage2<E, T, false>(X[c], j, [&](int q, int jj) { return Q[(q * T + jj) * Y2 + ln]; });
  }
  {
    float2* __restrict__ dst = (NC == 2 || comp1 == 0) ? g.m0 : (comp1 == 1 ? g.m1 : g.m2);
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int kx = j + T * r;
      float2 o;
      if constexpr (NC == 2) {
        const float kap = s_kx[kx];
        o = make_float2(-kap * X[0][r].y - kyv * X[1][r].y, kap * X[0][r].x + kyv * X[1][r].x);    // i kx J~x + i ky J~y
      } else {
        o = X[0][r];
        if (comp1 < 2) {
          const float kap = (comp1 == 0) ? s_kx[kx] : kyv;
          o = make_float2(-kap * o.y, kap * o.x);
        }
      }
      dst[((size_t)kx * nz + z) * Y2 + ln] = o;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// plane_unit3<N, E, EMIT>: ALL THREE components of plane z in one pass of a group (N <= 64): V~ and E~z are read
// once, the three transforms run interleaved between shared barriers, D~ = i kx J~x + i ky J~y and J~z leave as two
// arrays (m0, m2).  One exchange buffer per component (PlaneCfg<N>::BUF float2 each, at P0 + c BUF), reused in place:
// a barrier separates the last read of an exchange from the first write of the next.
// With nz plane units for about as many groups the plane phase is a single round.
// ------------------------------------------------------------------------------------------------
template <int N, int E, bool EMIT>
__device__ __forceinline__ void plane_unit3(const GeomDev& g, int nz, int z, const float2 (&VV)[E], const float2 (&VE)[E], float2* P0,
                                            const float* s_sdt, const float* s_kx, int tid, int bar_id, int slot) {
  using C = PlaneCfg<N>;
  constexpr int Y2 = C::Y2, T = N / E, SX = C::SX, SU = C::SU, NT = N * N / (2 * E), BUF = C::BUF, NC = 3;
  const int ln = tid % Y2, j = tid / Y2;
  float2 w[E];
  load_twiddles<E>(w, g.twx, j);
  unsigned short sid[E];
  if (!EMIT) {
    const unsigned short* st = reinterpret_cast<const unsigned short*>(g.sig_t + (size_t)z * N * N);
#pragma unroll
    for (int r = 0; r < E; ++r) sid[r] = __ldg(st + ((j + T * r) * N + 2 * ln) / 2);
  }
  const float kyv = __ldg(g.kyf + ln);
  float2 X[NC][E];
#pragma unroll
  for (int r = 0; r < E; ++r) {
    const float2 v = VV[r];
    const float kx = s_kx[j + T * r];
    X[0][r] = make_float2(kx * v.y, -kx * v.x);        // -i kx V~
    X[1][r] = make_float2(kyv * v.y, -kyv * v.x);      // -i ky V~
    X[2][r] = VE[r];                                   // E~z
  }
  // ---- A: inverse transform along x
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
    fft_stage1<E, true>(X[c], w);
#pragma unroll
    for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
    fft_stage2<E, T, true>(X[c], j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
#pragma unroll
    for (int r = 0; r < E; ++r) P[ln * SX + j + T * r] = X[c][r];        // transposed: [ky][x]
  }
  group_sync(bar_id, NT);
  // Hermitian completion along y of the two packed real rows (Nyquist = 0)
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      if (r < E / 2) {
        const float4 ab = *reinterpret_cast<const float4*>(&P[(j + T * r) * SX + 2 * ln]);
        X[c][r] = make_float2(ab.x - ab.w, ab.y + ab.z);
      } else {
        const int km = N - (j + T * r);
        if (km == Y2) {
          X[c][r] = make_float2(0.f, 0.f);
        } else {
          const float4 ab = *reinterpret_cast<const float4*>(&P[km * SX + 2 * ln]);
          X[c][r] = make_float2(ab.x + ab.w, ab.z - ab.y);
        }
      }
    }
    fft_stage1<E, true>(X[c], w);           // B: inverse transform along y
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
#pragma unroll
    for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
    fft_stage2<E, T, true>(X[c], j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
  }
  if constexpr (EMIT) {
    // (a8) H[n] = E/dt into the staging slot [slot][comp][z][y][x]
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      float2* st = reinterpret_cast<float2*>(g.stage + (((size_t)slot * 3 + c) * nz + z) * (size_t)(N * N));
#pragma unroll
      for (int r = 0; r < E; ++r) st[((j + T * r) * N + 2 * ln) / 2] = make_float2(X[c][r].x * g.inv_dt, X[c][r].y * g.inv_dt);
    }
    group_sync(bar_id, NT);                     // the buffers are rewritten by the group's next unit
    return;
  }
  // ---- J = (s dt_int) E nodewise (a6); C: forward transform along y
#pragma unroll
  for (int c = 0; c < NC; ++c) {
#pragma unroll
    for (int r = 0; r < E; ++r) {
      X[c][r].x *= s_sdt[sid[r] & 0xff];
      X[c][r].y *= s_sdt[sid[r] >> 8];
    }
    fft_stage1<E, false>(X[c], w);
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
#pragma unroll
    for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
    fft_stage2<E, T, false>(X[c], j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
#pragma unroll
    for (int r = 0; r < E; ++r) P[(j + T * r) * SU + ln] = X[c][r];      // [k][p2]
  }
  group_sync(bar_id, NT);
  // unpack the two real rows' half spectra; D: forward transform along x
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
    const int km = (N - ln) % N;
    const bool odd = j & 1;
#pragma unroll
    for (int r = 0; r < E; ++r) {
      const int p2 = (j + T * r) >> 1;
      const float2 zk = P[ln * SU + p2], zm = P[km * SU + p2];
      X[c][r] = odd ? make_float2(0.5f * (zk.y + zm.y), 0.5f * (zm.x - zk.x))
                    : make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
    }
    fft_stage1<E, false>(X[c], w);
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
#pragma unroll
    for (int q = 0; q < E; ++q) P[(q * T + j) * Y2 + ln] = X[c][q];
  }
  group_sync(bar_id, NT);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    float2* P = P0 + c * BUF;
    fft_stage2<E, T, false>(X[c], j, [&](int q, int jj) { return P[(q * T + jj) * Y2 + ln]; });
  }
#pragma unroll
  for (int r = 0; r < E; ++r) {
    const int kx = j + T * r;
    const float kap = s_kx[kx];
    const size_t o = ((size_t)kx * nz + z) * Y2 + ln;
    g.m0[o] = make_float2(-kap * X[0][r].y - kyv * X[1][r].y, kap * X[0][r].x + kyv * X[1][r].x);    // i kx J~x + i ky J~y
    g.m2[o] = X[2][r];
  }
  group_sync(bar_id, NT);                       // the buffers are rewritten by the group's next unit
}

// shared memory of one z-line group (transient part).  `red` (partial pad-layer sums, written after the per-mode
// update), `accp` (pad contributions, RES mode) and `cs` (charges times e^{-i kx x}, pass B) lie over `buf`
// (exchange buffer of the transforms), which is dead whenever they are live.
template <int NZ, int E, int TYL> struct ZGroupSmem {
  using C = PencilCfg<NZ, E, TYL>;
  static constexpr size_t buf = 0;                                                   // float2 [2][E][QS]
  static constexpr size_t buf_bytes = (size_t)2 * C::FIELD * sizeof(float2);
  static constexpr size_t red_bytes = (size_t)kMaxLayers * TYL * 2 * C::T * sizeof(double2);
  static constexpr size_t kzb = (buf_bytes > red_bytes ? buf_bytes : red_bytes);     // float2 [2][NZ][TYL]
  static constexpr size_t pls = kzb + (size_t)2 * NZ * TYL * sizeof(float2);         // double2 [kMaxLayers][TYL]
  static constexpr size_t bytes = pls + (size_t)kMaxLayers * TYL * sizeof(double2);
  static constexpr size_t state_bytes = (size_t)NZ * TYL * sizeof(double2);          // RES: the tile's fp64 charge spectrum
  static constexpr size_t gtab_bytes = (size_t)2 * NZ * TYL * sizeof(float);         // RES: the tile's slices of g~, g~_z at the head of buf during pass B
  static_assert(gtab_bytes + 1100 * sizeof(float2) <= buf_bytes, "g slices + charge factors must fit in the exchange buffer");
  static constexpr int max_pads = (int)(kzb / 16);                                    // cs[B] double2 must fit over buf
};

constexpr double kFixScale = 4398046511104.0;            // 2^42: pad potentials are accumulated as int64 fixed point
constexpr double kFixInv = 1.0 / 4398046511104.0;        // (integer adds commute: the sum over the CTAs is order independent)

// ------------------------------------------------------------------------------------------------
// z_pass_a: forward z DFT of (D~, J~z), per-mode Euler update of the fp64 state, V^_rho, pad-layer potentials of
// this tile (fp64) and their contribution to V_rho at every pad node (added to acc_pad).
// Thread mapping of k_pencil2 (solve_fast.cuh): (f, line, j), 2 * TYL * NZ/E threads.
//   RES   the group owns this one tile for the whole launch: its state lives in shared memory (rsm), the inverse
//         Green factors gg in registers, and V^_rho stays in kzb for z_pass_b
// ------------------------------------------------------------------------------------------------
template <int NZ, int E, int TYL, int LT, bool RES, bool MERGED, bool APPLY_J, bool DELTA>
__device__ __forceinline__ void z_pass_a(const PersistArgs& a, int tile, unsigned char* gsm, double2* rsm, const double (&gg)[E / 2],
                                         const double* s_kz, const float* s_kzf, const double2* s_twz, const double2* s_twx, const double2* s_twy,
                                         const int* s_px, const int* s_py, const int* s_pl, double* acc_pad, int tid, int bar_id) {
  using C = PencilCfg<NZ, E, TYL>;
  using S = ZGroupSmem<NZ, E, TYL>;
  constexpr int T = C::T, QS = C::QS, FIELD = C::FIELD, HT = C::THREADS, NT = 2 * HT;
  const GeomDev& g = a.g;
  const int nx = a.gd.nx, ny = a.gd.ny, y2 = a.gd.y2;
  const int tiles = y2 / TYL;
  const int kx = tile / tiles, ky0 = (tile % tiles) * TYL;
  const int f = tid / HT, th = tid % HT;
  const int line = th % TYL, j = th / TYL;
  const int ky = ky0 + line;
  const int L = g.L;
  float2* buf = reinterpret_cast<float2*>(gsm + S::buf) + f * FIELD;
  float2* kzb = reinterpret_cast<float2*>(gsm + S::kzb);
  double2* red = reinterpret_cast<double2*>(gsm + S::buf);
  double2* pls = reinterpret_cast<double2*>(gsm + S::pls);
  const size_t slab = (size_t)kx * NZ * y2 + ky;

  FSTAMP(0);
  if constexpr (APPLY_J) {
    float2 w[E];
    load_twiddles<E>(w, g.twz, j);
    float2 X[E];
    {
      const float2* __restrict__ mf = (f == 0 ? g.m0 : g.m2) + slab;      // D~ = i kx J~x + i ky J~y | J~z
#pragma unroll
      for (int r = 0; r < E; ++r) X[r] = ldcg2(mf + (size_t)(j + T * r) * y2);
      if (!MERGED && f == 0) {                                            // (plane phase with one component per unit: m0 + m1)
        const float2* __restrict__ m1 = g.m1 + slab;
#pragma unroll
        for (int r = 0; r < E; ++r) { const float2 q = ldcg2(m1 + (size_t)(j + T * r) * y2); X[r].x += q.x; X[r].y += q.y; }
      }
    }
    FSTAMP(1);
    fft_stage1<E, false>(X, w);
#pragma unroll
    for (int q = 0; q < E; ++q) buf[q * QS + j * TYL + line] = X[q];
    group_sync(bar_id, NT);
    FSTAMP(2);
    fft_stage2<E, T, false>(X, j, [&](int q, int jj) { return buf[q * QS + jj * TYL + line]; });
#pragma unroll
    for (int p = 0; p < E; ++p) kzb[(f * NZ + j + T * p) * TYL + line] = X[p];
    group_sync(bar_id, NT);
    FSTAMP(3);
  }
  {
    double2 acc[LT];
#pragma unroll
    for (int l = 0; l < LT; ++l) acc[l] = make_double2(0.0, 0.0);
    const double kxd = g.kxd[kx], kyd = g.kyd[ky];
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
      double2 rr = RES ? rsm[kz * TYL + line] : rh[o];
      if constexpr (APPLY_J) {
        const float2 D = kzb[kz * TYL + line], J = kzb[(NZ + kz) * TYL + line];
        const float kzf = s_kzf[kz];
        rr.x -= (double)(D.x - kzf * J.y);
        rr.y -= (double)(D.y + kzf * J.x);
        if (!ret) rr = make_double2(0.0, 0.0);
        if (RES) rsm[kz * TYL + line] = rr; else rh[o] = rr;
      }
      double2 src = rr;
      if constexpr (DELTA) {
        const double2 p = rp[o];
        src.x -= p.x; src.y -= p.y;
        if (RES) rp[o] = rr;                   // (two-pass mode: z_pass_b reads the old value once more and then writes)
      }
      double ggi;
      if constexpr (RES) {
        ggi = gg[i];
      } else {
        const double k2 = kxy2 + kzd * kzd;
        ggi = (ret && k2 > 0.0) ? a.gd.inv_n * fast_rcp(k2) : 0.0;
      }
      const double2 v = make_double2(src.x * ggi, src.y * ggi);
      if constexpr (RES) {                     // V^_rho and -i kz V^_rho wait in kzb for the boundary charges
        const float2 vf = make_float2((float)v.x, (float)v.y);
        const float kzf = s_kzf[kz];
        kzb[kz * TYL + line] = vf;
        kzb[(NZ + kz) * TYL + line] = make_float2(kzf * vf.y, -kzf * vf.x);
      }
#pragma unroll
      for (int l = 0; l < LT; ++l) {
        if (l < L) {
          if (g.layers[l] == 0) {                                                 // e^{+i kz 0} = 1
            acc[l].x += v.x; acc[l].y += v.y;
          } else {
            const double2 w = s_twz[(kz * g.layers[l]) & (NZ - 1)];               // acc += v e^{+i kz z_l} = v conj(w)
            acc[l].x = fma(v.x, w.x, fma(v.y, w.y, acc[l].x));
            acc[l].y = fma(v.y, w.x, fma(-v.x, w.y, acc[l].y));
          }
        }
      }
    }
#pragma unroll
    for (int l = 0; l < LT; ++l)
      if (l < L) red[(l * TYL + line) * (2 * T) + f * T + j] = acc[l];
  }
  group_sync(bar_id, NT);
  FSTAMP(4);
  // V~_rho(kx, z_l, ky) in fp64: 16 lanes per sum, fixed order (two terms per lane, then a shuffle tree)
  for (int i0 = 0; i0 < L * TYL; i0 += NT / 16) {
    const int i = i0 + tid / 16, sub = tid & 15;
    double2 s = make_double2(0.0, 0.0);
    if (i < L * TYL) {
      for (int k = sub; k < 2 * T; k += 16) { const double2 p = red[i * (2 * T) + k]; s.x += p.x; s.y += p.y; }
    }
#pragma unroll
    for (int d = 8; d > 0; d >>= 1) { s.x += __shfl_xor_sync(0xffffffffu, s.x, d); s.y += __shfl_xor_sync(0xffffffffu, s.y, d); }
    if (i < L * TYL && sub == 0) {
      const double wgt = (ky0 + i % TYL == 0) ? 1.0 : 2.0;          // Hermitian half spectrum along y
      pls[i] = make_double2(wgt * s.x, wgt * s.y);
    }
  }
  group_sync(bar_id, NT);
  FSTAMP(5);
  // contribution of this tile to V_rho at every pad node: Re( e^{+i kx x_b} sum_ky pl[l_b][ky] e^{+i ky y_b} )
  for (int b = tid; b < g.B; b += NT) {
    const int l = s_pl[b], y = s_py[b];
    double2 u0 = make_double2(0.0, 0.0), u1 = make_double2(0.0, 0.0);
#pragma unroll
    for (int ln = 0; ln < TYL; ln += 2) {
      const double2 p0 = dmulc(pls[l * TYL + ln], s_twy[((ky0 + ln) * y) & (ny - 1)]);
      const double2 p1 = dmulc(pls[l * TYL + ln + 1], s_twy[((ky0 + ln + 1) * y) & (ny - 1)]);
      u0.x += p0.x; u0.y += p0.y; u1.x += p1.x; u1.y += p1.y;
    }
    const double2 wx = s_twx[(kx * s_px[b]) & (nx - 1)];
    const double c = (u0.x + u1.x) * wx.x + (u0.y + u1.y) * wx.y;
    if (RES) acc_pad[b] = c; else acc_pad[b] += c;
  }
  FSTAMP(6);
}

// ------------------------------------------------------------------------------------------------
// z_pass_b: V^ = V^_rho + (sum_l S_l e^{-i kz z_l}) / |kappa|^2 with S_l(kx, ky) = sum_{b in l} Q'_b e^{-i(kx x_b + ky y_b)}
// the spectrum of the boundary point charges (a4: the translated fundamental solutions of PAPER.md:97 summed in
// spectral space), -i kz V^, inverse z DFTs -> (oV, oE).  RES: V^_rho waits in kzb (fp32) and the source is added in
// fp32; otherwise V^ is formed again from the fp64 state with the source added in fp64.
// ------------------------------------------------------------------------------------------------
template <int NZ, int E, int TYL, int LT, bool RES, bool DELTA>
__device__ __forceinline__ void z_pass_b(const PersistArgs& a, int tile, unsigned char* gsm, const double (&gg)[E / 2], const double* s_kz,
                                         const float* s_kzf, const float2* s_twzf, const float2* s_twxf, const float2* s_twyf, const double2* s_twz, const double2* s_twx, const double2* s_twy, const int* s_px, const int* s_py,
                                         float2* __restrict__ oV, float2* __restrict__ oE, int tid, int bar_id) {
  using C = PencilCfg<NZ, E, TYL>;
  using S = ZGroupSmem<NZ, E, TYL>;
  constexpr int T = C::T, QS = C::QS, FIELD = C::FIELD, HT = C::THREADS, NT = 2 * HT;
  const GeomDev& g = a.g;
  const int nx = a.gd.nx, ny = a.gd.ny, y2 = a.gd.y2;
  const int tiles = y2 / TYL;
  const int kx = tile / tiles, ky0 = (tile % tiles) * TYL;
  const int f = tid / HT, th = tid % HT;
  const int line = th % TYL, j = th / TYL;
  const int ky = ky0 + line;
  const int L = g.L, B = g.B;
  float2* buf = reinterpret_cast<float2*>(gsm + S::buf) + f * FIELD;
  float2* kzb = reinterpret_cast<float2*>(gsm + S::kzb);
  double2* cs = reinterpret_cast<double2*>(gsm + S::buf);        // [B] Q'_b e^{-i kx x_b}
  double2* pls = reinterpret_cast<double2*>(gsm + S::pls);       // reused: S_l(kx, ky0 + line)
  const size_t slab = (size_t)kx * NZ * y2 + ky;
  FSTAMP(8);
  if constexpr (RES) {
    // the spectrum of the charges is added in fp32 below: sums of <= a few hundred terms in fp32
    float2* csf = reinterpret_cast<float2*>(gsm + S::buf);       // [B] Q'_b e^{-i kx x_b}
    float2* plf = reinterpret_cast<float2*>(pls);                // [L][TYL] S_l(kx, ky0 + line)
    for (int b = tid; b < B; b += NT) {
      const float q = (float)__ldcg(g.q + b);
      const float2 wx = s_twxf[(kx * s_px[b]) & (nx - 1)];
      csf[b] = make_float2(q * wx.x, q * wx.y);
    }
    group_sync(bar_id, NT);
    for (int i0 = 0; i0 < L * TYL; i0 += NT / 16) {
      const int i = i0 + tid / 16, sub = tid & 15;
      float2 s0 = make_float2(0.f, 0.f), s1 = make_float2(0.f, 0.f);
      if (i < L * TYL) {
        const int l = i / TYL, kyy = ky0 + i - l * TYL;
        int b = a.lpoff[l] + sub;
        const int be = a.lpoff[l + 1];
        for (; b + 16 < be; b += 32) {
          const float2 c0 = csf[b], w0 = s_twyf[(kyy * s_py[b]) & (ny - 1)];
          const float2 c1 = csf[b + 16], w1 = s_twyf[(kyy * s_py[b + 16]) & (ny - 1)];
          s0.x += c0.x * w0.x - c0.y * w0.y; s0.y += c0.x * w0.y + c0.y * w0.x;
          s1.x += c1.x * w1.x - c1.y * w1.y; s1.y += c1.x * w1.y + c1.y * w1.x;
        }
        if (b < be) {
          const float2 c0 = csf[b], w0 = s_twyf[(kyy * s_py[b]) & (ny - 1)];
          s0.x += c0.x * w0.x - c0.y * w0.y; s0.y += c0.x * w0.y + c0.y * w0.x;
        }
      }
      float2 sv = make_float2(s0.x + s1.x, s0.y + s1.y);
#pragma unroll
      for (int d = 8; d > 0; d >>= 1) { sv.x += __shfl_xor_sync(0xffffffffu, sv.x, d); sv.y += __shfl_xor_sync(0xffffffffu, sv.y, d); }
      if (i < L * TYL && sub == 0) plf[i] = sv;
    }
  } else {
  for (int b = tid; b < B; b += NT) {
    const double q = __ldcg(g.q + b);
    const double2 wx = s_twx[(kx * s_px[b]) & (nx - 1)];
    cs[b] = make_double2(q * wx.x, q * wx.y);
  }
  group_sync(bar_id, NT);
  // S_l(kx, ky): 16 lanes per sum over the pads of the layer, fixed order
  for (int i0 = 0; i0 < L * TYL; i0 += NT / 16) {
    const int i = i0 + tid / 16, sub = tid & 15;
    double2 s = make_double2(0.0, 0.0);
    if (i < L * TYL) {
      const int l = i / TYL, ln = i - l * TYL;
      for (int b = a.lpoff[l] + sub; b < a.lpoff[l + 1]; b += 16) {
        const double2 p = dmul(cs[b], s_twy[((ky0 + ln) * s_py[b]) & (ny - 1)]);
        s.x += p.x; s.y += p.y;
      }
    }
#pragma unroll
    for (int d = 8; d > 0; d >>= 1) { s.x += __shfl_xor_sync(0xffffffffu, s.x, d); s.y += __shfl_xor_sync(0xffffffffu, s.y, d); }
    if (i < L * TYL && sub == 0) pls[i] = s;
  }
  }
  group_sync(bar_id, NT);
  FSTAMP(9);
  if constexpr (RES) {
    // the source in fp32: kzb += (sum_l S_l e^{-i kz z_l}) gg, and the same times -i kz
    const float2* plf = reinterpret_cast<const float2*>(pls);
    float2 sl[LT];
#pragma unroll
    for (int l = 0; l < LT; ++l) sl[l] = (l < L) ? plf[l * TYL + line] : make_float2(0.f, 0.f);
#pragma unroll
    for (int i = 0; i < E / 2; ++i) {
      const int kz = j + T * (2 * i + f);
      float2 src = make_float2(0.f, 0.f);
#pragma unroll
      for (int l = 0; l < LT; ++l) {
        if (l < L) {
          const float2 wz = s_twzf[(kz * g.layers[l]) & (NZ - 1)];
          src.x += sl[l].x * wz.x - sl[l].y * wz.y; src.y += sl[l].x * wz.y + sl[l].y * wz.x;
        }
      }
      const float gf = (float)gg[i], kzf = s_kzf[kz];
      const float2 v = make_float2(src.x * gf, src.y * gf);
      float2 c0 = kzb[kz * TYL + line], c1 = kzb[(NZ + kz) * TYL + line];
      c0.x += v.x; c0.y += v.y;
      c1.x += kzf * v.y; c1.y -= kzf * v.x;
      kzb[kz * TYL + line] = c0;
      kzb[(NZ + kz) * TYL + line] = c1;
    }
  } else {
    const double kxd = g.kxd[kx], kyd = g.kyd[ky];
    const double kxy2 = kxd * kxd + kyd * kyd;
    const bool ret_x = (kx != nx / 2);
    const double2* __restrict__ rh = g.rhat + slab;
    double2* __restrict__ rp = g.rhat_prev + slab;
#pragma unroll
    for (int i = 0; i < E / 2; ++i) {
      const int kz = j + T * (2 * i + f);
      const size_t o = (size_t)kz * y2;
      const bool ret = ret_x && (kz != NZ / 2);
      const double kzd = s_kz[kz];
      const double2 rr = rh[o];
      double2 src = rr;
      if constexpr (DELTA) {
        const double2 p = rp[o];
        src.x -= p.x; src.y -= p.y;
        rp[o] = rr;
      }
#pragma unroll
      for (int l = 0; l < LT; ++l) {
        if (l < L) {
          const double2 p = dmul(pls[l * TYL + line], s_twz[(kz * g.layers[l]) & (NZ - 1)]);   // S_l e^{-i kz z_l}
          src.x += p.x; src.y += p.y;
        }
      }
      const double k2 = kxy2 + kzd * kzd;
      const double ggi = (ret && k2 > 0.0) ? a.gd.inv_n * fast_rcp(k2) : 0.0;
      const double2 v = make_double2(src.x * ggi, src.y * ggi);
      kzb[kz * TYL + line] = make_float2((float)v.x, (float)v.y);
      kzb[(NZ + kz) * TYL + line] = make_float2((float)(kzd * v.y), (float)(-kzd * v.x));   // -i kz V^
    }
  }
  group_sync(bar_id, NT);
  FSTAMP(10);
  float2 w[E];
  load_twiddles<E>(w, g.twz, j);
  float2 X[E];
#pragma unroll
  for (int r = 0; r < E; ++r) X[r] = kzb[(f * NZ + j + T * r) * TYL + line];
  fft_stage1<E, true>(X, w);
#pragma unroll
  for (int q = 0; q < E; ++q) buf[q * QS + j * TYL + line] = X[q];
  group_sync(bar_id, NT);
  FSTAMP(11);
  fft_stage2<E, T, true>(X, j, [&](int q, int jj) { return buf[q * QS + jj * TYL + line]; });
  {
    float2* __restrict__ out = (f == 0 ? oV : oE) + slab;
#pragma unroll
    for (int r = 0; r < E; ++r) out[(size_t)(j + T * r) * y2] = X[r];
  }
  FSTAMP(12);
  group_sync(bar_id, NT);      // buf / kzb / pls are rewritten by the group's next tile
  FSTAMP(13);
}

// ------------------------------------------------------------------------------------------------
// RES only: pass B in two parts around the wait for the boundary charges.
//   z_pass_b_early  (while the boundary CTAs work)  inverse z DFTs of V^_rho and -i kz V^_rho, which wait in kzb, into the
//                   thread's own slots of kzb (field f at z = j + T r)
//   z_pass_b_late   (charges arrived)  S_l(kx, ky) = sum_{b in l} Q'_b e^{-i(kx x_b + ky y_b)} as in z_pass_b, then the boundary
//                   source in MIXED space, X += sum_l (S_l / N) g~(kx, z - z_l, ky)  (a4: the translated fundamental solutions
//                   of PAPER.md:97; the same sum the kernel chain forms in its plane kernel; z_pass_b_early fetched the tile's
//                   slices of g~, g~_z into shared memory meanwhile), and the store
// The transform no longer waits for the charges: about 3 us per substep leave the exposed chain at configs[1].
// ------------------------------------------------------------------------------------------------
template <int NZ, int E, int TYL, int LT>
__device__ __forceinline__ void z_pass_b_early(const PersistArgs& a, int tile, unsigned char* gsm, float2 (&X)[E], int tid, int bar_id) {
  using C = PencilCfg<NZ, E, TYL>;
  using S = ZGroupSmem<NZ, E, TYL>;
  constexpr int T = C::T, QS = C::QS, FIELD = C::FIELD, HT = C::THREADS, NT = 2 * HT;
  const GeomDev& g = a.g;
  const int y2 = a.gd.y2;
  const int tiles = y2 / TYL;
  const int kx = tile / tiles, ky0 = (tile % tiles) * TYL;
  const int f = tid / HT, th = tid % HT;
  const int line = th % TYL, j = th / TYL;
  float2* buf = reinterpret_cast<float2*>(gsm + S::buf) + f * FIELD;
  const float2* kzb = reinterpret_cast<const float2*>(gsm + S::kzb);
  float2 w[E];
  load_twiddles<E>(w, g.twz, j);
#pragma unroll
  for (int r = 0; r < E; ++r) X[r] = kzb[(f * NZ + j + T * r) * TYL + line];
  fft_stage1<E, true>(X, w);
#pragma unroll
  for (int q = 0; q < E; ++q) buf[q * QS + j * TYL + line] = X[q];
  group_sync(bar_id, NT);
  fft_stage2<E, T, true>(X, j, [&](int q, int jj) { return buf[q * QS + jj * TYL + line]; });
  // the transformed fields wait in the thread's own kzb slots (registers held across the wait spill at 128 per thread)
  float2* kzw = reinterpret_cast<float2*>(gsm + S::kzb);
#pragma unroll
  for (int r = 0; r < E; ++r) kzw[(f * NZ + j + T * r) * TYL + line] = X[r];
  group_sync(bar_id, NT);      // (all reads of the exchange buffer done)
  // the tile's slices of the mixed-space fundamental solution g~(kx, dz, ky), g~_z to the head of buf: static tables, so the
  // loads fly while the boundary CTAs work; z_pass_b_late adds the boundary source from them
  float* sg = reinterpret_cast<float*>(gsm + S::buf);
  for (int i = tid; i < 2 * NZ * TYL; i += NT) {
    const int ff = i / (NZ * TYL), rem = i - ff * (NZ * TYL), dz = rem / TYL, ln = rem - dz * TYL;
    sg[i] = __ldg((ff == 0 ? g.gt : g.gzt) + ((size_t)kx * NZ + dz) * y2 + ky0 + ln);
  }
}

template <int NZ, int E, int TYL, int LT>
__device__ __forceinline__ void z_pass_b_late(const PersistArgs& a, int tile, unsigned char* gsm, float2 (&X)[E], const float2* s_twxf, const float2* s_twyf, const int* s_px, const int* s_py,
                                              float2* __restrict__ oV, float2* __restrict__ oE, int tid, int bar_id) {
  using C = PencilCfg<NZ, E, TYL>;
  using S = ZGroupSmem<NZ, E, TYL>;
  constexpr int T = C::T, HT = C::THREADS, NT = 2 * HT;
  const GeomDev& g = a.g;
  const int nx = a.gd.nx, ny = a.gd.ny, y2 = a.gd.y2;
  const int tiles = y2 / TYL;
  const int kx = tile / tiles, ky0 = (tile % tiles) * TYL;
  const int f = tid / HT, th = tid % HT;
  const int line = th % TYL, j = th / TYL;
  const int L = g.L, B = g.B;
  const float* s_g = reinterpret_cast<const float*>(gsm + S::buf);                   // [2][NZ][TYL], written by z_pass_b_early
  float2* csf = reinterpret_cast<float2*>(gsm + S::buf + S::gtab_bytes);             // [B] Q'_b e^{-i kx x_b}
  float2* plf = reinterpret_cast<float2*>(gsm + S::pls);       // [L][TYL] S_l(kx, ky0 + line)
  for (int b = tid; b < B; b += NT) {
    const float q = (float)__ldcg(g.q + b);
    const float2 wx = s_twxf[(kx * s_px[b]) & (nx - 1)];
    csf[b] = make_float2(q * wx.x, q * wx.y);
  }
  group_sync(bar_id, NT);
  for (int i0 = 0; i0 < L * TYL; i0 += NT / 16) {
    const int i = i0 + tid / 16, sub = tid & 15;
    float2 s0 = make_float2(0.f, 0.f), s1 = make_float2(0.f, 0.f);
    if (i < L * TYL) {
      const int l = i / TYL, kyy = ky0 + i - l * TYL;
      int b = a.lpoff[l] + sub;
      const int be = a.lpoff[l + 1];
      for (; b + 16 < be; b += 32) {
        const float2 c0 = csf[b], w0 = s_twyf[(kyy * s_py[b]) & (ny - 1)];
        const float2 c1 = csf[b + 16], w1 = s_twyf[(kyy * s_py[b + 16]) & (ny - 1)];
        s0.x += c0.x * w0.x - c0.y * w0.y; s0.y += c0.x * w0.y + c0.y * w0.x;
        s1.x += c1.x * w1.x - c1.y * w1.y; s1.y += c1.x * w1.y + c1.y * w1.x;
      }
      if (b < be) {
        const float2 c0 = csf[b], w0 = s_twyf[(kyy * s_py[b]) & (ny - 1)];
        s0.x += c0.x * w0.x - c0.y * w0.y; s0.y += c0.x * w0.y + c0.y * w0.x;
      }
    }
    float2 sv = make_float2(s0.x + s1.x, s0.y + s1.y);
#pragma unroll
    for (int d = 8; d > 0; d >>= 1) { sv.x += __shfl_xor_sync(0xffffffffu, sv.x, d); sv.y += __shfl_xor_sync(0xffffffffu, sv.y, d); }
    if (i < L * TYL && sub == 0) plf[i] = sv;
  }
  group_sync(bar_id, NT);
  const float inv_n = (float)a.gd.inv_n;
  const float* __restrict__ tab = s_g + (size_t)f * NZ * TYL + line;      // the tile's g~ (f = 0) or g~_z (f = 1), [dz][TYL]
  {
    const float2* kzr = reinterpret_cast<const float2*>(gsm + S::kzb);
#pragma unroll
    for (int r = 0; r < E; ++r) X[r] = kzr[(f * NZ + j + T * r) * TYL + line];
  }
#pragma unroll
  for (int l = 0; l < LT; ++l) {
    if (l < L) {
      const float2 sl = make_float2(plf[l * TYL + line].x * inv_n, plf[l * TYL + line].y * inv_n);
#pragma unroll
      for (int r = 0; r < E; ++r) {
        const float t = tab[((j + T * r - g.layers[l]) & (NZ - 1)) * TYL];
        X[r].x = fmaf(sl.x, t, X[r].x); X[r].y = fmaf(sl.y, t, X[r].y);
      }
    }
  }
  {
    float2* __restrict__ out = (f == 0 ? oV : oE) + (size_t)kx * NZ * y2 + ky0 + line;
#pragma unroll
    for (int r = 0; r < E; ++r) out[(size_t)(j + T * r) * y2] = X[r];
  }
  group_sync(bar_id, NT);      // buf / kzb / pls are rewritten by the group's next phase
}

// ------------------------------------------------------------------------------------------------
// The kernel.  grid = n_z_cta + n_b_cta CTAs of kPersistThreads threads (cooperative launch: all resident).
// Dynamic shared memory: [tables][transient phase region][persistent region: fp64 state of the CTA's tiles (Z CTAs,
// RES) | rhs, V_pad and the CTA's rows of Ainv (B CTAs)].
// ------------------------------------------------------------------------------------------------
template <int N, int EP, int NZ, int EZ, int TYL> struct PersistCfg {
  static constexpr int PT = N * N / (2 * EP);                       // threads of a plane group
  static constexpr int ZT = 2 * PencilCfg<NZ, EZ, TYL>::THREADS;    // threads of a z-line group
  static constexpr int PG = kPersistThreads / PT, ZG = kPersistThreads / ZT;
  static_assert(PG >= 1 && ZG >= 1 && PG <= 8 && ZG <= 8, "group sizes");
  static constexpr bool MERGED = (N <= 64);                        // plane units carry the x and y components together
  static constexpr size_t p_bytes = (size_t)PG * (MERGED ? 3 : 2) * PlaneCfg<N>::BUF * sizeof(float2);
  static constexpr size_t z_bytes = (size_t)ZG * ZGroupSmem<NZ, EZ, TYL>::bytes;
  static constexpr size_t t_bytes = (size_t)4 * kStageSlots * 3 * N * sizeof(float);   // transpose phase: four (z, y) units in flight
  static constexpr size_t phase_bytes = (p_bytes > z_bytes ? p_bytes : z_bytes) > t_bytes ? (p_bytes > z_bytes ? p_bytes : z_bytes) : t_bytes;
  static constexpr size_t state_bytes = (size_t)ZG * ZGroupSmem<NZ, EZ, TYL>::state_bytes;
};

struct PersistSmem {        // byte offsets of the table section (host and device agree through this function)
  size_t kz, kzf, twz, twzf, twx, twy, twxf, twyf, px, py, pl, acc, sdt, kxf, phase;
};
// acc_groups: z-line groups that need their own pad accumulators in the table section (0 in RES mode)
__host__ __device__ inline PersistSmem persist_smem(int nx, int ny, int nz, int B, int acc_groups) {
  PersistSmem s;
  size_t p = 0;
  auto take = [&](size_t b) { size_t at = p; p = (p + b + 15) / 16 * 16; return at; };
  s.kz = take((size_t)nz * 8); s.kzf = take((size_t)nz * 4); s.twz = take((size_t)nz * 16); s.twzf = take((size_t)nz * 8);
  s.twx = take((size_t)nx * 16); s.twy = take((size_t)ny * 16); s.twxf = take((size_t)nx * 8); s.twyf = take((size_t)ny * 8);
  s.px = take((size_t)B * 4); s.py = take((size_t)B * 4); s.pl = take((size_t)B * 4);
  s.acc = take((size_t)acc_groups * B * 8);
  s.sdt = take(256 * 4); s.kxf = take((size_t)nx * 4);
  s.phase = p;
  return s;
}

template <int N, int EP, int NZ, int EZ, int TYL, int LT, bool RES>
__global__ void __launch_bounds__(kPersistThreads, 1) k_persistent(const __grid_constant__ PersistArgs a) {
  using CF = PersistCfg<N, EP, NZ, EZ, TYL>;
  using ZS = ZGroupSmem<NZ, EZ, TYL>;
  constexpr int PT = CF::PT, ZT = CF::ZT, PG = CF::PG, ZG = CF::ZG;
  constexpr int TZ = NZ / EZ;
  const GeomDev& g = a.g;
  PersistCtl* ctl = a.ctl;
  if (*reinterpret_cast<volatile int*>(&ctl->abort)) return;
  const int tid = threadIdx.x, cta = blockIdx.x, n_cta = gridDim.x;
  const int B = g.B, Bs = g.Bs;
  const int nx = N, ny = N, y2 = N / 2, nz = NZ;
  extern __shared__ __align__(16) unsigned char smraw[];
  const PersistSmem so = persist_smem(nx, ny, nz, B, RES ? 0 : ZG);
  double* s_kz = reinterpret_cast<double*>(smraw + so.kz);
  double2* s_twz = reinterpret_cast<double2*>(smraw + so.twz);
  float* s_kzf = reinterpret_cast<float*>(smraw + so.kzf);
  float2* s_twzf = reinterpret_cast<float2*>(smraw + so.twzf);
  float2* s_twxf = reinterpret_cast<float2*>(smraw + so.twxf);
  float2* s_twyf = reinterpret_cast<float2*>(smraw + so.twyf);
  double2* s_twx = reinterpret_cast<double2*>(smraw + so.twx);
  double2* s_twy = reinterpret_cast<double2*>(smraw + so.twy);
  int* s_px = reinterpret_cast<int*>(smraw + so.px);
  int* s_py = reinterpret_cast<int*>(smraw + so.py);
  int* s_pl = reinterpret_cast<int*>(smraw + so.pl);
  float* s_sdt = reinterpret_cast<float*>(smraw + so.sdt);
  float* s_kxf = reinterpret_cast<float*>(smraw + so.kxf);
  unsigned char* phase = smraw + so.phase;
  unsigned char* persist = smraw + a.smem_persist_off;
  // B CTAs: rhs [Bs], V_pad [Bs], rows of Ainv
  double* s_rhs = reinterpret_cast<double*>(persist);
  double* s_vpad = s_rhs + Bs;
  double* s_ainv = s_vpad + Bs;
  __shared__ int s_ok;

  const bool is_z = cta < a.n_z_cta;
  const int brank = cta - a.n_z_cta;                       // rank among the B CTAs (>= 0 for them)
  const int rows_per = (B + a.n_b_cta - 1) / a.n_b_cta;
  const int r0 = is_z ? 0 : min(B, brank * rows_per), r1 = is_z ? 0 : min(B, r0 + rows_per);
  const int n_tiles = nx * (y2 / TYL);

  for (int i = tid; i < nz; i += kPersistThreads) { s_kz[i] = g.kzd[i]; s_twz[i] = g.twzd[i]; s_kzf[i] = g.kzf[i]; s_twzf[i] = g.twz[i]; }
  for (int i = tid; i < nx; i += kPersistThreads) { s_twx[i] = g.twxd[i]; s_kxf[i] = g.kxf[i]; s_twxf[i] = g.twx[i]; }
  for (int i = tid; i < ny; i += kPersistThreads) { s_twy[i] = g.twyd[i]; s_twyf[i] = g.twy[i]; }
  for (int i = tid; i < 256; i += kPersistThreads) s_sdt[i] = g.sdt[i];
  for (int i = tid; i < B; i += kPersistThreads) { s_px[i] = a.pad_x[i]; s_py[i] = g.pad_y[i]; s_pl[i] = a.pad_l[i]; }
  if (!is_z) {
    for (int i = tid; i < B; i += kPersistThreads) s_vpad[i] = g.pad_pot[i];
    if (a.ainv_in_smem)
      for (int i = tid; i < (r1 - r0) * Bs; i += kPersistThreads) s_ainv[i] = g.ainv[(size_t)r0 * Bs + i];
  }
  // RES: the group's tile, its fp64 state (shared memory) and inverse Green factors (registers) for the whole launch
  const int zgrp = tid / ZT, zt = tid % ZT;
  const int my_tile = cta + a.n_z_cta * zgrp;
  double2* rsm = reinterpret_cast<double2*>(persist + (size_t)zgrp * ZS::state_bytes);
  double gg[EZ / 2];
#pragma unroll
  for (int i = 0; i < EZ / 2; ++i) gg[i] = 0.0;
  if (RES && is_z && my_tile < n_tiles) {
    const int tiles = y2 / TYL;
    const int kx = my_tile / tiles, ky0 = (my_tile % tiles) * TYL;
    constexpr int HT = ZT / 2;
    const int f = zt / HT, th = zt % HT, line = th % TYL, j = th / TYL;
    const double kxd = g.kxd[kx], kyd = g.kyd[ky0 + line];
#pragma unroll
    for (int i = 0; i < EZ / 2; ++i) {
      const int kz = j + TZ * (2 * i + f);
      const double kzd = g.kzd[kz];
      const double k2 = kxd * kxd + kyd * kyd + kzd * kzd;
      gg[i] = (kx != nx / 2 && kz != NZ / 2 && k2 > 0.0) ? a.gd.inv_n / k2 : 0.0;
    }
    for (int i = zt; i < NZ * TYL; i += ZT) {
      const int kz = i / TYL, ln = i - kz * TYL;
      rsm[i] = g.rhat[((size_t)kx * NZ + kz) * y2 + ky0 + ln];
    }
  }
  __syncthreads();

#ifdef WTIDE_DEBUG
  int n_stamp = 0;
  auto stamp = [&]() {
    if (a.stamps && a.step == 2 && tid == 0 && n_stamp < 28) {
      unsigned long long t;
      asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
      a.stamps[(size_t)cta * 64 + n_stamp++] = t;
    }
  };
#define PSTAMP() stamp()
#else
#define PSTAMP() do { } while (0)
#endif
  unsigned long long bar_n = a.bar0, epi = a.epi0;
  auto grid_barrier = [&]() -> bool {
    cta_signal(&ctl->bar);
    ++bar_n;
    return cta_wait(&ctl->bar, bar_n * (unsigned long long)n_cta, &ctl->abort, &s_ok);
  };

  // ---- phases ---------------------------------------------------------------------------------
  auto plane_phase = [&](auto emit_tag, const float2* srcV, const float2* srcE, int slot) {
    constexpr bool EMIT = decltype(emit_tag)::value;
    // units: nz "xy" units (components x and y of a plane together, twice the work) first, then nz "z" units
    const int grp = tid / PT, t = tid % PT;
    const int n_slots = n_cta * PG;
    if constexpr (CF::MERGED) {
      // one unit = all three components of a plane: nz units for n_cta * PG groups (a single round at configs[1])
      float2 VV[EP], VE[EP];
      float2* P0 = reinterpret_cast<float2*>(phase) + (size_t)grp * 3 * PlaneCfg<N>::BUF;
      for (int u = cta * PG + grp; u < nz; u += n_slots) {
        plane_load<N, EP>(VV, srcV, nz, u, t);
        plane_load<N, EP>(VE, srcE, nz, u, t);
        plane_unit3<N, EP, EMIT>(g, nz, u, VV, VE, P0, s_sdt, s_kxf, t, 1 + grp, slot);
      }
    } else {
      float2* P0 = reinterpret_cast<float2*>(phase) + (size_t)grp * 2 * PlaneCfg<N>::BUF;
      float2 V[EP];
      for (int u = cta * PG + grp; u < nz * 3; u += n_slots) {
        const int z = u / 3, comp = u - 3 * z;
        plane_load<N, EP>(V, comp == 2 ? srcE : srcV, nz, z, t);
        plane_unit<N, EP, EMIT, 1>(g, nz, z, comp, V, P0, s_sdt, s_kxf, t, 1 + grp, slot);
      }
    }
  };
  // z-line phase incl. the boundary adjust; flag = 1: pads at their potentials, 0: homogeneous (increment)
  auto z_phase = [&](auto apply_tag, auto delta_tag, double flag, float2* oV, float2* oE) -> bool {
    constexpr bool APPLY_J = decltype(apply_tag)::value;
    constexpr bool DELTA = decltype(delta_tag)::value;
    ++epi;
    long long* fix = a.fix + (size_t)(epi & 1ULL) * Bs;            // this episode's fixed-point pad potentials
    if (is_z) {
      unsigned char* gsm = phase + (size_t)zgrp * ZS::bytes;
      double* acc = RES ? reinterpret_cast<double*>(gsm + ZS::buf) : reinterpret_cast<double*>(smraw + so.acc) + (size_t)zgrp * B;
      if (!RES) {
        for (int b = zt; b < B; b += ZT) acc[b] = 0.0;
        group_sync(1 + zgrp, ZT);
      }
      bool any = false;
      for (int tile = my_tile; tile < n_tiles; tile += a.n_z_cta * ZG) {
        z_pass_a<NZ, EZ, TYL, LT, RES, CF::MERGED, APPLY_J, DELTA>(a, tile, gsm, rsm, gg, s_kz, s_kzf, s_twz, s_twx, s_twy, s_px, s_py, s_pl, acc, zt, 1 + zgrp);
        any = true;
      }
      if (RES && !any)
        for (int b = zt; b < B; b += ZT) acc[b] = 0.0;
      __syncthreads();
      PSTAMP();   // z1: pass A done
      for (int b = tid; b < B; b += kPersistThreads) {
        double s = 0.0;
#pragma unroll
        for (int q = 0; q < ZG; ++q)
          s += RES ? reinterpret_cast<const double*>(phase + (size_t)q * ZS::bytes + ZS::buf)[b] : reinterpret_cast<const double*>(smraw + so.acc)[(size_t)q * B + b];
        atomicAdd(reinterpret_cast<unsigned long long*>(fix + b), (unsigned long long)__double2ll_rn(s * kFixScale));
      }
      cta_signal(&ctl->cnt_part);
      PSTAMP();   // z2: contributions published
      if constexpr (RES) {
        // the group's one tile: the inverse transform runs while the boundary CTAs solve for the charges
        float2 XB[EZ];
        const bool have = my_tile < n_tiles;
        if (have) z_pass_b_early<NZ, EZ, TYL, LT>(a, my_tile, gsm, XB, zt, 1 + zgrp);
        if (!cta_wait(&ctl->cnt_q, epi * (unsigned long long)a.n_b_cta, &ctl->abort, &s_ok)) return false;
        PSTAMP();   // z3: charges arrived
        if (have) z_pass_b_late<NZ, EZ, TYL, LT>(a, my_tile, gsm, XB, s_twxf, s_twyf, s_px, s_py, oV, oE, zt, 1 + zgrp);
      } else {
        if (!cta_wait(&ctl->cnt_q, epi * (unsigned long long)a.n_b_cta, &ctl->abort, &s_ok)) return false;
        PSTAMP();   // z3: charges arrived
        for (int tile = my_tile; tile < n_tiles; tile += a.n_z_cta * ZG)
          z_pass_b<NZ, EZ, TYL, LT, RES, DELTA>(a, tile, gsm, gg, s_kz, s_kzf, s_twzf, s_twxf, s_twyf, s_twz, s_twx, s_twy, s_px, s_py, oV, oE, zt, 1 + zgrp);
      }
      PSTAMP();   // z4: pass B done
    } else {
      // ---- boundary adjust on the B CTAs: rows [r0, r1) --------------------------------------------
      const int warp = tid >> 5, lane = tid & 31;
      constexpr int kWarps = kPersistThreads / 32;
      long long* fix_next = a.fix + (size_t)((epi + 1) & 1ULL) * Bs;
      if (!cta_wait(&ctl->cnt_part, epi * (unsigned long long)a.n_z_cta, &ctl->abort, &s_ok)) return false;
      PSTAMP();   // b1: all contributions in
      for (int b = tid; b < B; b += kPersistThreads)          // rhs = flag V_pad - V_rho|_B, every B CTA the whole vector
        s_rhs[b] = flag * s_vpad[b] - (double)__ldcg(fix + b) * kFixInv;
      for (int b = r0 + tid; b < r1; b += kPersistThreads) fix_next[b] = 0;   // (read last in the previous episode)
      __syncthreads();
      PSTAMP();   // b2: rhs
      for (int row = r0 + warp; row < r1; row += kWarps) {     // Q' = Ainv rhs, one warp per row, fixed order
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        int jj = lane;
        if (a.ainv_in_smem) {
          const double* __restrict__ ar = s_ainv + (size_t)(row - r0) * Bs;
          for (; jj + 96 < B; jj += 128) {
            s0 += ar[jj] * s_rhs[jj]; s1 += ar[jj + 32] * s_rhs[jj + 32];
            s2 += ar[jj + 64] * s_rhs[jj + 64]; s3 += ar[jj + 96] * s_rhs[jj + 96];
          }
          for (; jj < B; jj += 32) s0 += ar[jj] * s_rhs[jj];
        } else {
          const double* __restrict__ ar = g.ainv + (size_t)row * Bs;
          for (; jj + 96 < B; jj += 128) {
            s0 += ar[jj] * s_rhs[jj]; s1 += ar[jj + 32] * s_rhs[jj + 32];
            s2 += ar[jj + 64] * s_rhs[jj + 64]; s3 += ar[jj + 96] * s_rhs[jj + 96];
          }
          for (; jj < B; jj += 32) s0 += ar[jj] * s_rhs[jj];
        }
        double s = (s0 + s1) + (s2 + s3);
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0) g.q[row] = s;
      }
      cta_signal(&ctl->cnt_q);
      PSTAMP();   // b3: charges published
      PSTAMP();   // (b4: keeps the stamp count equal to the z-line CTAs')
    }
    return true;
  };
  auto transpose_phase = [&](int n) {
    // staging [slot][comp][z][y][x] -> H[((x*ny+y)*nz+z)*nt + t][comp] for the last cnt output steps (k_transpose<true>)
    const int cnt = n % kStageSlots + 1, t0 = n - cnt + 1, rows = cnt * 3;
    float* tile = reinterpret_cast<float*>(phase);
    const int nt = a.gd.nt;
    auto run = [&](auto rows_c, auto u_c) {
      // U (z, y) units per round, `rows` a compile-time constant where it is the full staging group (index arithmetic by constants)
      constexpr int U = decltype(u_c)::value;
      const int rows_ = decltype(rows_c)::value ? decltype(rows_c)::value : rows;
      const int per = rows_ * nx;
      for (int unit0 = cta * U; unit0 < nz * ny; unit0 += n_cta * U) {
        const int nu = min(U, nz * ny - unit0);
        for (int t = tid; t < nu * per; t += kPersistThreads) {
          const int u = t / per, r = t - u * per;
          const int unit = unit0 + u, z = unit / ny, y = unit - z * ny;
          const int j = r / nx, x = r - j * nx;
          tile[t] = __ldcg(g.stage + (((size_t)j * nz + z) * ny + y) * nx + x);
        }
        __syncthreads();
        for (int t = tid; t < nu * per; t += kPersistThreads) {
          const int u = t / per, r = t - u * per;
          const int unit = unit0 + u, z = unit / ny, y = unit - z * ny;
          const int x = r / rows_, j = r - x * rows_;
          g.H[((((size_t)x * ny + y) * nz + z) * nt + t0) * 3 + j] = tile[u * per + j * nx + x];
        }
        __syncthreads();
      }
    };
    if (rows == 3 * kStageSlots) run(std::integral_constant<int, 3 * kStageSlots>{}, std::integral_constant<int, 4>{});
    else run(std::integral_constant<int, 0>{}, std::integral_constant<int, 1>{});
  };
  // RES: the state goes back to global memory for the next launch
  auto save_state = [&]() {
    if (RES && is_z && my_tile < n_tiles) {
      const int tiles = y2 / TYL;
      const int kx = my_tile / tiles, ky0 = (my_tile % tiles) * TYL;
      for (int i = zt; i < NZ * TYL; i += ZT) {
        const int kz = i / TYL, ln = i - kz * TYL;
        g.rhat[((size_t)kx * NZ + kz) * y2 + ky0 + ln] = rsm[i];
      }
    }
  };

  using TT = std::true_type;
  using FF = std::false_type;
  const int n = a.step;
  const int slot = n % kStageSlots;
  if (n == 0) {
    // prompt response: r = 0, pads at their potentials.  The same potential starts the step pipeline.
    if (!z_phase(FF{}, FF{}, 1.0, g.v0, g.v1)) return;
    if (!grid_barrier()) return;
    plane_phase(TT{}, g.v0, g.v1, slot);
  } else {
    for (int s = 0; s < a.n_sub; ++s) {
#ifdef WTIDE_DEBUG
      if (tid == 0) g_fine_on = (s == 1);
      __syncthreads();
#endif
      PSTAMP();   // p0: substep starts
      plane_phase(FF{}, g.v0, g.v1, 0);
      PSTAMP();   // p1: plane units done
      if (!grid_barrier()) return;
      PSTAMP();   // p2: barrier passed
      if (!z_phase(TT{}, FF{}, 1.0, g.v0, g.v1)) return;
      if (!grid_barrier()) return;
    }
    // H[n] from the increment of the charge since the previous output step, pads at 0 V
    if (!z_phase(FF{}, TT{}, 0.0, g.e0, g.e1)) return;
    save_state();
    if (!grid_barrier()) return;
    plane_phase(TT{}, g.e0, g.e1, slot);
  }
  if ((n + 1) % kStageSlots == 0 || n == a.gd.nt - 1) {
    if (!grid_barrier()) return;
    transpose_phase(n);
  }
}

// last launch of a persistent solve: a time-out anywhere poisons the table (the call is asynchronous: this is
// how the caller learns about it)
__global__ void k_persist_finish(PersistCtl* ctl, float* H) {
  if (ctl->abort) H[0] = __int_as_float(0x7fc00000);
}

}  // namespace wt
