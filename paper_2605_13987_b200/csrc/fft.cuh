// Shared-memory mixed-radix (8, 4, 2, 3) Stockham FFT building block for libwtide's spectral solve.
//
// PAPER.md:95 uses "the 3D FFT implementation shipped with CUDA" (cuFFT); here the 3-D transform is
// split into z-line and xy-plane kernels that keep a tile in shared memory and fuse the per-mode
// work around the 1-D passes.  This header holds the 1-D pass only.
//
// A "batch" is n_lines independent complex lines of length L living in shared memory; element i of
// line l sits at buf[l*ls + i*es].  Threads are mapped line-fastest, so accesses are bank-conflict
// free when ls == 1 or ls is odd.  Passes ping-pong between two buffers; every pass ends with
// __syncthreads().  Transforms are unnormalised; forward uses e^{-i}, inverse e^{+i}.
#pragma once
#include <cuda_runtime.h>

namespace wt {

template <typename C2> struct scalar_of;
template <> struct scalar_of<float2> { using type = float; };
template <> struct scalar_of<double2> { using type = double; };

template <typename C2> __device__ __forceinline__ C2 cmake(typename scalar_of<C2>::type x, typename scalar_of<C2>::type y) {
  C2 r; r.x = x; r.y = y; return r;
}
template <typename C2> __device__ __forceinline__ C2 cadd(C2 a, C2 b) { return cmake<C2>(a.x + b.x, a.y + b.y); }
template <typename C2> __device__ __forceinline__ C2 csub(C2 a, C2 b) { return cmake<C2>(a.x - b.x, a.y - b.y); }
template <typename C2> __device__ __forceinline__ C2 cmul(C2 a, C2 b) {
  return cmake<C2>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <typename C2> __device__ __forceinline__ C2 cconj(C2 a) { return cmake<C2>(a.x, -a.y); }
// multiply by -i (forward) or +i (inverse)
template <typename C2> __device__ __forceinline__ C2 crot(C2 a, bool inverse) {
  return inverse ? cmake<C2>(-a.y, a.x) : cmake<C2>(a.y, -a.x);
}

template <int R, typename C2> struct Butterfly;
template <typename C2> struct Butterfly<2, C2> {
  static __device__ __forceinline__ void run(C2* v, bool) {
    C2 a = v[0], b = v[1];
    v[0] = cadd(a, b); v[1] = csub(a, b);
  }
};
template <typename C2> struct Butterfly<4, C2> {
  static __device__ __forceinline__ void run(C2* v, bool inverse) {
    C2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
    C2 t2 = cadd(v[1], v[3]), t3 = crot(csub(v[1], v[3]), inverse);
    v[0] = cadd(t0, t2); v[1] = cadd(t1, t3); v[2] = csub(t0, t2); v[3] = csub(t1, t3);
  }
};
template <typename C2> struct Butterfly<8, C2> {
  // even / odd halves by two radix-4 butterflies, then X[k] = E[k] + W8^k O[k], X[k+4] = E[k] - W8^k O[k]
  static __device__ __forceinline__ void run(C2* v, bool inverse) {
    using T = typename scalar_of<C2>::type;
    const T h = (T)0.70710678118654752440;
    C2 e[4] = {v[0], v[2], v[4], v[6]}, o[4] = {v[1], v[3], v[5], v[7]};
    Butterfly<4, C2>::run(e, inverse);
    Butterfly<4, C2>::run(o, inverse);
    const T s = inverse ? (T)1 : (T)-1;            // W8 = (1 + s i)/sqrt(2)
    const C2 o1 = cmake<C2>(h * (o[1].x - s * o[1].y), h * (o[1].y + s * o[1].x));
    const C2 o2 = crot(o[2], inverse);
    const C2 o3 = cmake<C2>(h * (-o[3].x - s * o[3].y), h * (-o[3].y + s * o[3].x));   // W8^3 = (-1 + s i)/sqrt(2)
    v[0] = cadd(e[0], o[0]); v[4] = csub(e[0], o[0]);
    v[1] = cadd(e[1], o1);   v[5] = csub(e[1], o1);
    v[2] = cadd(e[2], o2);   v[6] = csub(e[2], o2);
    v[3] = cadd(e[3], o3);   v[7] = csub(e[3], o3);
  }
};
template <typename C2> struct Butterfly<3, C2> {
  static __device__ __forceinline__ void run(C2* v, bool inverse) {
    using T = typename scalar_of<C2>::type;
    const T h = (T)0.86602540378443864676;   // sqrt(3)/2
    C2 s = cadd(v[1], v[2]), d = csub(v[1], v[2]);
    C2 m = cmake<C2>(v[0].x - (T)0.5 * s.x, v[0].y - (T)0.5 * s.y);
    C2 n = crot(d, inverse);
    n.x *= h; n.y *= h;
    v[0] = cadd(v[0], s); v[1] = cadd(m, n); v[2] = csub(m, n);
  }
};

// One Stockham pass of radix R.  tw[k * tw_stride] = e^{-2 pi i k / L}, k < L.
template <int R, typename C2>
__device__ __forceinline__ void fft_pass(const C2* __restrict__ in, C2* __restrict__ out, int L, int Ns,
                                         int n_lines, int ls, int es, const C2* __restrict__ tw, bool inverse) {
  const int per_line = L / R;
  const int total = per_line * n_lines;
  const int tmul = L / (Ns * R);
  // t / n_lines by a multiply (exact for t * n_lines < 2^32, i.e. any tile that fits in shared memory);
  // j % Ns by a mask while Ns is a power of two (always, except after a first radix-3 pass)
  const unsigned inv_lines = 0xffffffffu / (unsigned)n_lines + 1u;
  const bool ns_pow2 = (Ns & (Ns - 1)) == 0;
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int j = (n_lines == 1) ? t : (int)__umulhi((unsigned)t, inv_lines), line = t - j * n_lines;
    const int k = ns_pow2 ? (j & (Ns - 1)) : j % Ns;
    const C2* src = in + line * ls;
    C2 v[R];
#pragma unroll
    for (int r = 0; r < R; ++r) v[r] = src[(j + r * per_line) * es];
    const int tstep = k * tmul;
#pragma unroll
    for (int r = 1; r < R; ++r) {
      C2 w = tw[r * tstep];
      if (inverse) w.y = -w.y;
      v[r] = cmul(v[r], w);
    }
    Butterfly<R, C2>::run(v, inverse);
    const int j0 = (j - k) * R + k;
    C2* dst = out + line * ls;
#pragma unroll
    for (int r = 0; r < R; ++r) dst[(j0 + r * Ns) * es] = v[r];
  }
  __syncthreads();
}

// Full 1-D transform of a batch.  Data must be visible (a __syncthreads() after it was written).
// Returns the buffer that holds the result (a or b); the other one is scratch.
template <typename C2>
__device__ __forceinline__ C2* fft_lines(C2* a, C2* b, int L, int n_lines, int ls, int es, const C2* __restrict__ tw,
                                         bool inverse) {
  int Ns = 1, rem = L;
  while (rem % 8 == 0) {
    fft_pass<8, C2>(a, b, L, Ns, n_lines, ls, es, tw, inverse);
    C2* t = a; a = b; b = t; Ns *= 8; rem /= 8;
  }
  while (rem % 4 == 0) {
    fft_pass<4, C2>(a, b, L, Ns, n_lines, ls, es, tw, inverse);
    C2* t = a; a = b; b = t; Ns *= 4; rem /= 4;
  }
  if (rem % 2 == 0) {
    fft_pass<2, C2>(a, b, L, Ns, n_lines, ls, es, tw, inverse);
    C2* t = a; a = b; b = t; Ns *= 2; rem /= 2;
  }
  while (rem % 3 == 0) {
    fft_pass<3, C2>(a, b, L, Ns, n_lines, ls, es, tw, inverse);
    C2* t = a; a = b; b = t; Ns *= 3; rem /= 3;
  }
  return a;
}

// number of passes fft_lines() runs for length L (parity of the ping-pong)
__host__ __device__ inline int fft_num_passes(int L) {
  int p = 0;
  while (L % 8 == 0) { ++p; L /= 8; }
  while (L % 4 == 0) { ++p; L /= 4; }
  if (L % 2 == 0) { ++p; L /= 2; }
  while (L % 3 == 0) { ++p; L /= 3; }
  return p;
}

}  // namespace wt
