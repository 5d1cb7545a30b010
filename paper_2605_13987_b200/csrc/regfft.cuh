// Register-resident FFT building blocks for libwtide's size-specialised solve kernels.
//
// PAPER.md:95 uses cuFFT for the 3-D transforms; libwtide splits them into z-line and xy-plane
// kernels.  For the power-of-two sizes of the BASELINE configs a line of
// length N is spread over T = N/E threads, each holding E elements in registers, and transformed
// by two Cooley-Tukey stages with ONE shared-memory exchange in between:
//
//   index split  n = j + T r  (j < T thread, r < E register),   k = q + E p  (q < E, p < T)
//   W_N^{nk} = W_E^{rq} . W_N^{jq} . W_T^{jp}
//   stage 1 (thread j):  Y_j[q] = W_N^{jq} sum_r x[j + T r] W_E^{rq}          (radix-E butterfly + twiddle)
//   exchange:            thread t collects Y_j[q] for q = t + T u (u < E/T), all j
//   stage 2 (thread t):  X[q + E p] = sum_j Y_j[q] W_T^{jp}                    (E/T radix-T butterflies)
//
// After stage 2 thread t holds X[t + T r'] with r' = u + (E/T) p: the same strided distribution
// as the input, so transforms chain without re-shuffling.  All indices are compile-time; the only
// run-time twiddles are the E per-thread factors W_N^{jq}, loaded once per kernel.
// Transforms are unnormalised; forward uses e^{-i}, inverse e^{+i}.
#pragma once
#include <cuda_runtime.h>

namespace wt {

__device__ __forceinline__ float2 c_add(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 c_sub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 c_mul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * conj(b)
__device__ __forceinline__ float2 c_mulc(float2 a, float2 b) {
  return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

// a * e^{-+ 2 pi i K/16}  (forward: minus, inverse: plus), K compile-time
template <int K, bool INV>
__device__ __forceinline__ float2 mul_w16(float2 a) {
  constexpr int k = ((K % 16) + 16) % 16;
  constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f, R = 0.70710678118654752f;
  // cos(2 pi k/16), sin(2 pi k/16)
  constexpr float cs[16] = {1.f, C1, R, S1, 0.f, -S1, -R, -C1, -1.f, -C1, -R, -S1, 0.f, S1, R, C1};
  constexpr float sn[16] = {0.f, S1, R, C1, 1.f, C1, R, S1, 0.f, -S1, -R, -C1, -1.f, -C1, -R, -S1};
  if constexpr (k == 0) return a;
  else if constexpr (k == 8) return make_float2(-a.x, -a.y);
  else if constexpr (k == 4) return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
  else if constexpr (k == 12) return INV ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
  else {
    constexpr float wr = cs[k];
    constexpr float wi = INV ? sn[k] : -sn[k];
    return make_float2(a.x * wr - a.y * wi, a.x * wi + a.y * wr);
  }
}

template <bool INV>
__device__ __forceinline__ void dft2(float2& a, float2& b) {
  const float2 s = c_add(a, b), d = c_sub(a, b);
  a = s; b = d;
}

// natural order in, natural order out
template <bool INV>
__device__ __forceinline__ void dft4(float2& v0, float2& v1, float2& v2, float2& v3) {
  const float2 t0 = c_add(v0, v2), t1 = c_sub(v0, v2);
  const float2 t2 = c_add(v1, v3), t3 = mul_w16<4, INV>(c_sub(v1, v3));
  v0 = c_add(t0, t2); v1 = c_add(t1, t3); v2 = c_sub(t0, t2); v3 = c_sub(t1, t3);
}

template <bool INV>
__device__ __forceinline__ void dft8(float2 (&v)[8]) {
  // even / odd halves, then X[k] = E[k] + W8^k O[k], X[k+4] = E[k] - W8^k O[k]
  dft4<INV>(v[0], v[2], v[4], v[6]);
  dft4<INV>(v[1], v[3], v[5], v[7]);
  const float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
  const float2 o0 = v[1], o1 = mul_w16<2, INV>(v[3]), o2 = mul_w16<4, INV>(v[5]), o3 = mul_w16<6, INV>(v[7]);
  v[0] = c_add(e0, o0); v[4] = c_sub(e0, o0);
  v[1] = c_add(e1, o1); v[5] = c_sub(e1, o1);
  v[2] = c_add(e2, o2); v[6] = c_sub(e2, o2);
  v[3] = c_add(e3, o3); v[7] = c_sub(e3, o3);
}

template <bool INV>
__device__ __forceinline__ void dft16(float2 (&v)[16]) {
  // n = 4a + b, k = c + 4d:  W16^{nk} = W4^{ac} W16^{bc} W4^{bd}
  dft4<INV>(v[0], v[4], v[8], v[12]);    // b = 0: Y_0[c] in v[4c]
  dft4<INV>(v[1], v[5], v[9], v[13]);    // b = 1: Y_1[c] in v[4c+1]
  dft4<INV>(v[2], v[6], v[10], v[14]);
  dft4<INV>(v[3], v[7], v[11], v[15]);
  // twiddle Y_b[c] *= W16^{bc}
  v[5] = mul_w16<1, INV>(v[5]);   v[9] = mul_w16<2, INV>(v[9]);   v[13] = mul_w16<3, INV>(v[13]);
  v[6] = mul_w16<2, INV>(v[6]);   v[10] = mul_w16<4, INV>(v[10]); v[14] = mul_w16<6, INV>(v[14]);
  v[7] = mul_w16<3, INV>(v[7]);   v[11] = mul_w16<6, INV>(v[11]); v[15] = mul_w16<9, INV>(v[15]);
  // for each c: X[c + 4d] = sum_b Y_b[c] W4^{bd}; Y_b[c] sits in v[4c + b]
  dft4<INV>(v[0], v[1], v[2], v[3]);     // c = 0 -> X[0], X[4], X[8], X[12] in v[0..3]
  dft4<INV>(v[4], v[5], v[6], v[7]);     // c = 1 -> X[1], X[5], X[9], X[13] in v[4..7]
  dft4<INV>(v[8], v[9], v[10], v[11]);
  dft4<INV>(v[12], v[13], v[14], v[15]);
  // v[4c + d] holds X[c + 4d]: transpose the 4x4 register tile into natural order
  float2 t;
  t = v[1]; v[1] = v[4]; v[4] = t;
  t = v[2]; v[2] = v[8]; v[8] = t;
  t = v[3]; v[3] = v[12]; v[12] = t;
  t = v[6]; v[6] = v[9]; v[9] = t;
  t = v[7]; v[7] = v[13]; v[13] = t;
  t = v[11]; v[11] = v[14]; v[14] = t;
}

// ---- radix 3 (grids 96 = 2^5 3, 384 = 2^7 3 of BASELINE configs[4]) -------------------------------------------
// a * e^{-+ 2 pi i K/24}  (forward: minus, inverse: plus), K compile-time
template <int K, bool INV>
__device__ __forceinline__ float2 mul_w24(float2 a) {
  constexpr int k = ((K % 24) + 24) % 24;
  constexpr float C1 = 0.96592582628906829f, C2 = 0.86602540378443865f, C3 = 0.70710678118654752f, C4 = 0.5f, C5 = 0.25881904510252076f;
  // cos(2 pi k/24), sin(2 pi k/24), k = 0 .. 23 (steps of 15 degrees)
  constexpr float cs[24] = {1.f, C1, C2, C3, C4, C5, 0.f, -C5, -C4, -C3, -C2, -C1, -1.f, -C1, -C2, -C3, -C4, -C5, 0.f, C5, C4, C3, C2, C1};
  constexpr float sn[24] = {0.f, C5, C4, C3, C2, C1, 1.f, C1, C2, C3, C4, C5, 0.f, -C5, -C4, -C3, -C2, -C1, -1.f, -C1, -C2, -C3, -C4, -C5};
  if constexpr (k == 0) return a;
  else if constexpr (k == 12) return make_float2(-a.x, -a.y);
  else if constexpr (k == 6) return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
  else if constexpr (k == 18) return INV ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
  else {
    constexpr float wr = cs[k];
    constexpr float wi = INV ? sn[k] : -sn[k];
    return make_float2(a.x * wr - a.y * wi, a.x * wi + a.y * wr);
  }
}

// X0 = a + b + c,  X1 = a + b w + c w^2,  X2 = a + b w^2 + c w,  w = e^{-+ 2 pi i/3}
template <bool INV>
__device__ __forceinline__ void dft3(float2& a, float2& b, float2& c) {
  constexpr float h = 0.86602540378443865f;   // sqrt(3)/2
  const float2 s = c_add(b, c), d = c_sub(b, c);
  const float2 m = make_float2(a.x - 0.5f * s.x, a.y - 0.5f * s.y);
  const float2 n = INV ? make_float2(-h * d.y, h * d.x) : make_float2(h * d.y, -h * d.x);   // (+-i) h d
  a = c_add(a, s); b = c_add(m, n); c = c_sub(m, n);
}

template <int B, int C, bool INV> struct Twiddle24 {
  static __device__ __forceinline__ void run(float2 (&y)[3][8]) {
    y[B][C] = mul_w24<B * C, INV>(y[B][C]);
    if constexpr (C + 1 < 8) Twiddle24<B, C + 1, INV>::run(y);
    else if constexpr (B + 1 < 3) Twiddle24<B + 1, 1, INV>::run(y);
  }
};

// n = 3a + b (a < 8, b < 3), k = c + 8d (c < 8, d < 3):  W24^{nk} = W8^{ac} W24^{bc} W3^{bd};  natural order in and out
template <bool INV>
__device__ __forceinline__ void dft24(float2 (&v)[24]) {
  float2 y[3][8];
#pragma unroll
  for (int b = 0; b < 3; ++b) {
#pragma unroll
    for (int a = 0; a < 8; ++a) y[b][a] = v[3 * a + b];
    dft8<INV>(y[b]);                          // Y_b[c]
  }
  Twiddle24<1, 1, INV>::run(y);               // Y_b[c] *= W24^{bc}
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    dft3<INV>(y[0][c], y[1][c], y[2][c]);     // d = 0, 1, 2
    v[c] = y[0][c]; v[c + 8] = y[1][c]; v[c + 16] = y[2][c];
  }
}

template <int R, bool INV>
__device__ __forceinline__ void dft(float2 (&v)[R]) {
  static_assert(R == 2 || R == 4 || R == 8 || R == 16 || R == 24, "radix");
  if constexpr (R == 2) dft2<INV>(v[0], v[1]);
  else if constexpr (R == 4) dft4<INV>(v[0], v[1], v[2], v[3]);
  else if constexpr (R == 8) dft8<INV>(v);
  else if constexpr (R == 16) dft16<INV>(v);
  else dft24<INV>(v);
}

// Per-thread twiddles w[q] = e^{-2 pi i j q/N}, q < E, from a table tw[k] = e^{-2 pi i k/N} (k < N).
template <int E>
__device__ __forceinline__ void load_twiddles(float2 (&w)[E], const float2* __restrict__ tw, int j) {
#pragma unroll
  for (int q = 0; q < E; ++q) w[q] = __ldg(tw + j * q);
}

// stage 1: radix-E butterfly over the thread's registers, then the twiddle W_N^{jq}
template <int E, bool INV>
__device__ __forceinline__ void fft_stage1(float2 (&v)[E], const float2 (&w)[E]) {
  dft<E, INV>(v);
#pragma unroll
  for (int q = 1; q < E; ++q) v[q] = INV ? c_mulc(v[q], w[q]) : c_mul(v[q], w[q]);
}

// the same with the twiddles read from a table (shared memory) where E registers for them are too many
template <int E, bool INV>
__device__ __forceinline__ void fft_stage1(float2 (&v)[E], const float2* __restrict__ w) {
  dft<E, INV>(v);
#pragma unroll
  for (int q = 1; q < E; ++q) v[q] = INV ? c_mulc(v[q], w[q]) : c_mul(v[q], w[q]);
}

// stage 2: thread t gathers Y_j[q] through `at(q, j)`, q = t + T u, and leaves X[t + T r'] in
// v[r'], r' = u + (E/T) p.
template <int E, int T, bool INV, typename At>
__device__ __forceinline__ void fft_stage2(float2 (&v)[E], int t, At at) {
  static_assert(E % T == 0, "E must be a multiple of T");
  constexpr int U = E / T;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    float2 y[T];
    const int q = t + T * u;
#pragma unroll
    for (int j = 0; j < T; ++j) y[j] = at(q, j);
    dft<T, INV>(y);
#pragma unroll
    for (int p = 0; p < T; ++p) v[u + U * p] = y[p];
  }
}

}  // namespace wt
