// SURVEY 8(f) rows 2 and 3 around the hot path: the static weighting field of a table, saturated-drift carrier
// transport in it (the step the paper says now dominates the time-to-insight) feeding Eq. 1.1
// without leaving HBM, and the electronics stage (transfer function of the front end, noise).
//
// Transport arithmetic is fp32 in a fixed order WITHOUT FMA contraction (explicit __fmul_rn / __fadd_rn ...), so
// that step counts -- decided by float comparisons -- and positions equal the oracle's bit for bit (R35).
#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "geometry.h"
#include "locate.cuh"

namespace {
using wt::locate;
using wt::NodeFrac;

constexpr int kMaxCols = 127;

struct DriftParams {
  const float* es;          // [nx*ny*nz][3]
  const float* start;       // [C][3]
  const int8_t* sign;       // [C]
  int64_t n_carriers;
  int nx, ny, nz, max_steps, n_cols;
  float invx, invy, invz, lx, ly, lz, dt, v_bias, mu_e, mu_h, v_sat;
  const float* cols;        // [n_cols][3] = (cx, cy, r*r) device
};

// Es[node][c] = dt * sum_n H[node][n][c]: one warp per node row (3 nt floats, 12 per lane and pass)
__global__ void __launch_bounds__(256) k_static_field(const float* __restrict__ H, float* __restrict__ es, int64_t n_nodes, int nt, float dt) {
  const int lane = threadIdx.x & 31;
  const int64_t node = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (node >= n_nodes) return;
  const float4* row = reinterpret_cast<const float4*>(H + (size_t)node * nt * 3);
  float sx = 0.f, sy = 0.f, sz = 0.f;
  for (int q = lane; 4 * q < nt; q += 32) {          // 4 time samples = 3 float4
    const float4 a = __ldg(row + 3 * q), b = __ldg(row + 3 * q + 1), c = __ldg(row + 3 * q + 2);
    sx += (a.x + a.w) + (b.z + c.y);
    sy += (a.y + b.x) + (b.w + c.z);
    sz += (a.z + b.y) + (c.x + c.w);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sx += __shfl_xor_sync(0xffffffffu, sx, o); sy += __shfl_xor_sync(0xffffffffu, sy, o); sz += __shfl_xor_sync(0xffffffffu, sz, o);
  }
  if (lane == 0) { es[3 * node] = sx * dt; es[3 * node + 1] = sy * dt; es[3 * node + 2] = sz * dt; }
}

__device__ __forceinline__ bool alive(float x, float y, float z, const DriftParams& p, const float* s_cols) {
  if (!(z >= 0.f && z <= p.lz)) return false;
  for (int c = 0; c < p.n_cols; ++c) {
    float dx = fmodf(fabsf(__fsub_rn(x, s_cols[3 * c])), p.lx);
    dx = fminf(dx, __fsub_rn(p.lx, dx));
    float dy = fmodf(fabsf(__fsub_rn(y, s_cols[3 * c + 1])), p.ly);
    dy = fminf(dy, __fsub_rn(p.ly, dy));
    if (!(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)) > s_cols[3 * c + 2])) return false;
  }
  return true;
}

// One thread per carrier.  FILL = false: counts[c] = number of recorded steps; FILL = true: pos / vel at offsets[c].
template <bool FILL>
__global__ void __launch_bounds__(128) k_drift(DriftParams p, int64_t* __restrict__ counts, const int64_t* __restrict__ offsets,
                                               float* __restrict__ pos, float* __restrict__ vel) {
  __shared__ float s_cols[3 * kMaxCols];
  for (int i = threadIdx.x; i < 3 * p.n_cols; i += blockDim.x) s_cols[i] = p.cols[i];
  __syncthreads();
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= p.n_carriers) return;
  float x = p.start[3 * c], y = p.start[3 * c + 1], z = p.start[3 * c + 2];
  const float sg = (float)p.sign[c];
  const float mu = sg < 0.f ? p.mu_e : p.mu_h;
  const float smu = __fmul_rn(sg, mu);
  int64_t o = FILL ? offsets[c] : 0;
  int m = 0;
  while (m < p.max_steps && isfinite(x) && isfinite(y) && isfinite(z) && alive(x, y, z, p, s_cols)) {
    const NodeFrac nf = locate(x, y, z, p.nx, p.ny, p.nz, p.invx, p.invy, p.invz);
    float ex = 0.f, ey = 0.f, ez = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const int cx = k >> 2, cy = (k >> 1) & 1, cz = k & 1;
      const float wx = cx ? nf.f[0] : __fsub_rn(1.f, nf.f[0]);
      const float wy = cy ? nf.f[1] : __fsub_rn(1.f, nf.f[1]);
      const float wz = cz ? nf.f[2] : __fsub_rn(1.f, nf.f[2]);
      const float w = __fmul_rn(__fmul_rn(wx, wy), wz);
      const int ix = cx ? nf.i1[0] : nf.i0[0], iy = cy ? nf.i1[1] : nf.i0[1], iz = cz ? nf.i1[2] : nf.i0[2];
      const float* e = p.es + 3 * ((size_t)(ix * p.ny + iy) * p.nz + iz);
      ex = __fadd_rn(ex, __fmul_rn(w, __ldg(e)));
      ey = __fadd_rn(ey, __fmul_rn(w, __ldg(e + 1)));
      ez = __fadd_rn(ez, __fmul_rn(w, __ldg(e + 2)));
    }
    ex = __fmul_rn(p.v_bias, ex); ey = __fmul_rn(p.v_bias, ey); ez = __fmul_rn(p.v_bias, ez);
    const float en = __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey)), __fmul_rn(ez, ez)));
    const float den = __fadd_rn(1.f, __fdiv_rn(__fmul_rn(mu, en), p.v_sat));
    const float vx = __fdiv_rn(__fmul_rn(smu, ex), den), vy = __fdiv_rn(__fmul_rn(smu, ey), den), vz = __fdiv_rn(__fmul_rn(smu, ez), den);
    const float xn = __fadd_rn(x, __fmul_rn(vx, p.dt)), yn = __fadd_rn(y, __fmul_rn(vy, p.dt)), zn = __fadd_rn(z, __fmul_rn(vz, p.dt));
    if (FILL) {
      pos[3 * o] = x; pos[3 * o + 1] = y; pos[3 * o + 2] = z;
      vel[3 * o] = __fdiv_rn(__fsub_rn(xn, x), p.dt); vel[3 * o + 1] = __fdiv_rn(__fsub_rn(yn, y), p.dt); vel[3 * o + 2] = __fdiv_rn(__fsub_rn(zn, z), p.dt);
      ++o;
    }
    x = xn; y = yn; z = zn;
    ++m;
  }
  if (!FILL) counts[c] = m;
}

// offsets[0] = 0, offsets[i + 1] = counts[0] + ... + counts[i]: one CTA, chunks of 1024 x 4 with a running carry
__global__ void __launch_bounds__(1024) k_offsets(const int64_t* __restrict__ counts, int64_t* __restrict__ offsets, int64_t n) {
  __shared__ int64_t s_warp[32];
  __shared__ int64_t s_carry;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) { s_carry = 0; offsets[0] = 0; }
  __syncthreads();
  for (int64_t base = 0; base < n; base += 4096) {
    int64_t v[4], t = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) { const int64_t k = base + 4 * tid + i; v[i] = k < n ? counts[k] : 0; t += v[i]; }
    int64_t incl = t;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int64_t u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      int64_t w = s_warp[lane], wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int64_t u = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += u; }
      s_warp[lane] = wi - w;                     // exclusive prefix of the warp totals
    }
    __syncthreads();
    int64_t run = s_carry + s_warp[warp] + (incl - t);
#pragma unroll
    for (int i = 0; i < 4; ++i) { const int64_t k = base + 4 * tid + i; run += v[i]; if (k < n) offsets[k + 1] = run; }
    __syncthreads();
    if (tid == 1023) s_carry = run;
    __syncthreads();
  }
}

// Electronics stage: one CTA per output row.  out[n] = dt sum_j h[j] cur[n - j] (+ noise[n]); constant-fraction time.
__global__ void __launch_bounds__(256) k_electronics(const float* __restrict__ cur, const float* __restrict__ h, int nh,
                                                     const float* __restrict__ noise, float dt, float frac, int nt, float* __restrict__ out,
                                                     float* __restrict__ t_cfd) {
  extern __shared__ float sm[];
  float* s_cur = sm;              // [nt]
  float* s_h = sm + nt;           // [nh]
  float* s_out = s_h + nh;        // [nt]
  __shared__ float s_val[256];
  __shared__ int s_idx[256];
  const int row = blockIdx.x, tid = threadIdx.x;
  for (int i = tid; i < nt; i += blockDim.x) s_cur[i] = cur[(size_t)row * nt + i];
  for (int i = tid; i < nh; i += blockDim.x) s_h[i] = h[i];
  __syncthreads();
  float best = -1.f;
  int best_i = 0x7fffffff;
  for (int n = tid; n < nt; n += blockDim.x) {
    float acc = 0.f;
    const int jm = min(nh, n + 1);
    for (int j = 0; j < jm; ++j) acc = fmaf(s_h[j], s_cur[n - j], acc);
    float v = acc * dt;
    if (noise) v += noise[(size_t)row * nt + n];
    s_out[n] = v;
    out[(size_t)row * nt + n] = v;
    if (fabsf(v) > best) { best = fabsf(v); best_i = n; }          // (ascending n per thread: first maximum kept)
  }
  s_val[tid] = best; s_idx[tid] = best_i;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {                                // extremum by absolute value, smallest index on ties
    if (tid < o) {
      const float v2 = s_val[tid + o];
      const int i2 = s_idx[tid + o];
      if (v2 > s_val[tid] || (v2 == s_val[tid] && i2 < s_idx[tid])) { s_val[tid] = v2; s_idx[tid] = i2; }
    }
    __syncthreads();
  }
  const int k = s_idx[0];
  const float peak = (k < nt) ? s_out[k] : 0.f;
  __syncthreads();
  if (peak == 0.f) { if (tid == 0) t_cfd[row] = -1.f; return; }
  const float s = peak > 0.f ? 1.f : -1.f, thr = frac * peak;
  int first = 0x7fffffff;
  for (int n = tid; n <= k; n += blockDim.x)
    if (s * s_out[n] >= s * thr) { first = n; break; }
  s_idx[tid] = first;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (tid < o) s_idx[tid] = min(s_idx[tid], s_idx[tid + o]);
    __syncthreads();
  }
  if (tid == 0) {
    const int n = s_idx[0];
    if (n == 0) t_cfd[row] = 0.f;
    else {
      const float a = s * s_out[n - 1], b = s * s_out[n];
      t_cfd[row] = (float)(n - 1) + (s * thr - a) / (b - a);
    }
  }
}

int fail(const char* fn, const std::string& msg, int code) { wt_set_error(std::string(fn) + ": " + msg); return code; }

}  // namespace

extern "C" int wt_static_field(const wt_geometry* g, const float* H_dev, float* es_dev, void* cuda_stream) {
  if (!wt_valid(g) || !H_dev || !es_dev || !cuda_stream) return fail("wt_static_field", "bad argument or NULL (default) stream", WT_EINVAL);
  if (((uintptr_t)H_dev) % 16 != 0) return fail("wt_static_field", "H table not 16-byte aligned", WT_EINVAL);
  const int64_t n_nodes = (int64_t)g->nx * g->ny * g->nz;
  ++g_wt_launches;
  k_static_field<<<(unsigned)((n_nodes + 7) / 8), 256, 0, (cudaStream_t)cuda_stream>>>(H_dev, es_dev, n_nodes, g->nt, (float)g->dt);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail("wt_static_field", cudaGetErrorString(e), WT_ECUDA);
  wt_set_error("");
  return WT_OK;
}

extern "C" int wt_drift_workspace_bytes(const wt_geometry* g, size_t* bytes) {
  if (!wt_valid(g) || !bytes) return fail("wt_drift_workspace_bytes", "bad argument", WT_EINVAL);
  *bytes = (size_t)3 * kMaxCols * sizeof(float) + 256;
  return WT_OK;
}

static int drift_call(bool fill, const wt_geometry* g, const float* es_dev, double v_bias, double mu_e, double mu_h, double v_sat,
                      int64_t n_carriers, const float* start_dev, const int8_t* sign_dev, int max_steps, int64_t* counts_dev,
                      const int64_t* offsets_dev, float* pos_dev, float* vel_dev, void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  const char* fn = fill ? "wt_drift_fill" : "wt_drift_count";
  if (!wt_valid(g) || !es_dev || !cuda_stream || n_carriers < 0 || max_steps < 0 || !workspace_dev)
    return fail(fn, "bad argument or NULL (default) stream", WT_EINVAL);
  if (n_carriers > 0 && (!start_dev || !sign_dev || (fill ? (!offsets_dev || !pos_dev || !vel_dev) : !counts_dev)))
    return fail(fn, "null array", WT_EINVAL);
  if (!(v_sat > 0) || !(mu_e > 0) || !(mu_h > 0)) return fail(fn, "mobilities and v_sat must be > 0", WT_EINVAL);
  size_t need = 0;
  wt_drift_workspace_bytes(g, &need);
  if (workspace_bytes < need) return fail(fn, "workspace too small", WT_ENOMEM);
  if ((int)g->cols_f32.size() > 3 * kMaxCols) return fail(fn, "too many columns", WT_EINVAL);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaMemcpyAsync(workspace_dev, g->cols_f32.data(), g->cols_f32.size() * sizeof(float), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail(fn, cudaGetErrorString(e), WT_ECUDA);
  DriftParams p;
  p.es = es_dev; p.start = start_dev; p.sign = sign_dev; p.n_carriers = n_carriers;
  p.nx = g->nx; p.ny = g->ny; p.nz = g->nz; p.max_steps = max_steps; p.n_cols = (int)g->cols_f32.size() / 3;
  p.invx = (float)((double)g->nx / g->lx); p.invy = (float)((double)g->ny / g->ly); p.invz = (float)((double)g->nz / g->lz);
  p.lx = (float)g->lx; p.ly = (float)g->ly; p.lz = (float)g->lz; p.dt = (float)g->dt;
  p.v_bias = (float)v_bias; p.mu_e = (float)mu_e; p.mu_h = (float)mu_h; p.v_sat = (float)v_sat;
  p.cols = (const float*)workspace_dev;
  if (n_carriers > 0) {
    ++g_wt_launches;
    const unsigned blocks = (unsigned)((n_carriers + 127) / 128);
    if (fill) k_drift<true><<<blocks, 128, 0, st>>>(p, nullptr, offsets_dev, pos_dev, vel_dev);
    else      k_drift<false><<<blocks, 128, 0, st>>>(p, counts_dev, nullptr, nullptr, nullptr);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(fn, cudaGetErrorString(e), WT_ECUDA);
  wt_set_error("");
  return WT_OK;
}

extern "C" int wt_drift_count(const wt_geometry* g, const float* es_dev, double v_bias, double mu_e, double mu_h, double v_sat,
                              int64_t n_carriers, const float* start_dev, const int8_t* sign_dev, int max_steps, int64_t* counts_dev,
                              void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  return drift_call(false, g, es_dev, v_bias, mu_e, mu_h, v_sat, n_carriers, start_dev, sign_dev, max_steps, counts_dev, nullptr, nullptr,
                    nullptr, workspace_dev, workspace_bytes, cuda_stream);
}

extern "C" int wt_drift_fill(const wt_geometry* g, const float* es_dev, double v_bias, double mu_e, double mu_h, double v_sat,
                             int64_t n_carriers, const float* start_dev, const int8_t* sign_dev, int max_steps,
                             const int64_t* carrier_step_offsets_dev, float* pos_dev, float* vel_dev, void* workspace_dev,
                             size_t workspace_bytes, void* cuda_stream) {
  return drift_call(true, g, es_dev, v_bias, mu_e, mu_h, v_sat, n_carriers, start_dev, sign_dev, max_steps, nullptr,
                    carrier_step_offsets_dev, pos_dev, vel_dev, workspace_dev, workspace_bytes, cuda_stream);
}

extern "C" int wt_offsets_from_counts(int64_t n, const int64_t* counts_dev, int64_t* offsets_dev, void* cuda_stream) {
  if (n < 0 || !offsets_dev || (n > 0 && !counts_dev) || !cuda_stream) return fail("wt_offsets_from_counts", "bad argument", WT_EINVAL);
  ++g_wt_launches;
  k_offsets<<<1, 1024, 0, (cudaStream_t)cuda_stream>>>(counts_dev, offsets_dev, n);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail("wt_offsets_from_counts", cudaGetErrorString(e), WT_ECUDA);
  wt_set_error("");
  return WT_OK;
}

extern "C" int wt_electronics(int64_t n_rows, int nt, const float* currents_dev, const float* transfer_dev, int n_transfer,
                              const float* noise_dev, double dt, double cfd_fraction, float* out_dev, float* t_cfd_dev, void* cuda_stream) {
  if (n_rows < 0 || nt < 1 || n_transfer < 1 || !cuda_stream || !transfer_dev || (n_rows > 0 && (!currents_dev || !out_dev || !t_cfd_dev)))
    return fail("wt_electronics", "bad argument or NULL (default) stream", WT_EINVAL);
  const size_t smem = ((size_t)2 * nt + n_transfer) * sizeof(float);
  if (smem > 200 * 1024) return fail("wt_electronics", "row + transfer function do not fit in shared memory", WT_EINVAL);
  if (n_rows > 0x7fffffffLL) return fail("wt_electronics", "too many rows", WT_EINVAL);
  cudaError_t e = cudaFuncSetAttribute(k_electronics, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return fail("wt_electronics", cudaGetErrorString(e), WT_ECUDA);
  if (n_rows > 0) {
    ++g_wt_launches;
    k_electronics<<<(unsigned)n_rows, 256, smem, (cudaStream_t)cuda_stream>>>(currents_dev, transfer_dev, n_transfer, noise_dev, (float)dt,
                                                                               (float)cfd_fraction, nt, out_dev, t_cfd_dev);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail("wt_electronics", cudaGetErrorString(e), WT_ECUDA);
  wt_set_error("");
  return WT_OK;
}
