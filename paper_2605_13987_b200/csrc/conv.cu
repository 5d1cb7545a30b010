// wt_convolve_currents / wt_trajectory_nodes: steps a9-a12 of the hot path (Eq. 1.1).
//
// PAPER.md:35-39 (Eq. 1.1), :74 ("for each charge carrier, the induced signal is computed as
// described in Equation 1.1"), :99 (one carrier per CUDA thread, H through texture interpolation).
// Here: one CTA per carrier, threads own output times n, the 8 corner rows of the time-innermost
// table are read with coalesced loads (consecutive threads = consecutive lags), trilinear weights
// in full fp32 (R23).  Per-track sums are formed in a second pass in carrier order (R25).
#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "geometry.h"

namespace {

struct ConvParams {
  const float* H;
  const int64_t* carrier_off;
  const float* pos;
  const float* vel;
  const float* charge;
  float* out;            // per-carrier rows [n_carriers][nt] (final output or workspace)
  int nx, ny, nz, nt;
  float invx, invy, invz;   // (float)((double)n / l)   (R24)
  float dt_over_vw;         // dt / v_w
};

struct NodeFrac {
  int i0[3], i1[3];
  float f[3];
  bool ok;
};

// R24: the index arithmetic of the ABI.  One fp32 multiply (no FMA contraction), floor, exact fraction.
__device__ __forceinline__ NodeFrac locate(float x, float y, float z, int nx, int ny, int nz, float invx, float invy,
                                           float invz) {
  NodeFrac r;
  r.ok = isfinite(x) && isfinite(y) && isfinite(z);
  if (!r.ok) {
    for (int a = 0; a < 3; ++a) { r.i0[a] = -1; r.i1[a] = -1; r.f[a] = 0.f; }
    return r;
  }
  const float ux = __fmul_rn(x, invx), uy = __fmul_rn(y, invy);
  float uz = __fmul_rn(z, invz);
  uz = fminf(fmaxf(uz, 0.f), (float)(nz - 1));
  const float fx = floorf(ux), fy = floorf(uy), fz = floorf(uz);
  r.f[0] = __fsub_rn(ux, fx); r.f[1] = __fsub_rn(uy, fy); r.f[2] = __fsub_rn(uz, fz);
  const long long ix = (long long)fx, iy = (long long)fy;
  const int iz = (int)fz;
  r.i0[0] = (int)(((ix % nx) + nx) % nx); r.i1[0] = (int)((((ix + 1) % nx) + nx) % nx);
  r.i0[1] = (int)(((iy % ny) + ny) % ny); r.i1[1] = (int)((((iy + 1) % ny) + ny) % ny);
  r.i0[2] = iz; r.i1[2] = min(iz + 1, nz - 1);
  return r;
}

constexpr int kThreads = 128;
constexpr int kOut = 4;      // outputs per thread per tile
constexpr int kChunk = 32;   // steps staged in shared memory at a time

// v1: one CTA per carrier; rows are read straight from global memory (L1/L2 give the reuse).
__global__ void __launch_bounds__(kThreads) k_conv_carrier(ConvParams p) {
  const int64_t c = blockIdx.x;
  const int64_t s0 = p.carrier_off[c];
  const int nt = p.nt;
  const int M = (int)min((int64_t)nt, p.carrier_off[c + 1] - s0);   // steps m >= nt are ignored (R26)
  const float scale = -p.charge[c] * p.dt_over_vw;
  __shared__ unsigned node[kChunk][8];
  __shared__ float coef[kChunk][8][3];
  const size_t row = (size_t)nt * 3;
  for (int n0 = 0; n0 < nt; n0 += kThreads * kOut) {
    float acc[kOut];
#pragma unroll
    for (int i = 0; i < kOut; ++i) acc[i] = 0.f;
    for (int m0 = 0; m0 < M; m0 += kChunk) {
      const int mc = min(kChunk, M - m0);
      __syncthreads();
      if ((int)threadIdx.x < mc) {
        const int64_t s = s0 + m0 + threadIdx.x;
        const float vx = p.vel[3 * s], vy = p.vel[3 * s + 1], vz = p.vel[3 * s + 2];
        NodeFrac nf = locate(p.pos[3 * s], p.pos[3 * s + 1], p.pos[3 * s + 2], p.nx, p.ny, p.nz, p.invx, p.invy, p.invz);
        const bool ok = nf.ok && isfinite(vx) && isfinite(vy) && isfinite(vz);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int cx = k >> 2, cy = (k >> 1) & 1, cz = k & 1;
          const float w = (cx ? nf.f[0] : 1.f - nf.f[0]) * (cy ? nf.f[1] : 1.f - nf.f[1]) * (cz ? nf.f[2] : 1.f - nf.f[2]);
          const int ix = cx ? nf.i1[0] : nf.i0[0], iy = cy ? nf.i1[1] : nf.i0[1], iz = cz ? nf.i1[2] : nf.i0[2];
          node[threadIdx.x][k] = ok ? (unsigned)((ix * p.ny + iy) * p.nz + iz) : 0u;
          const float ws = w * scale;     // a non-finite step contributes nothing (0, not 0 * inf)
          coef[threadIdx.x][k][0] = ok ? ws * vx : 0.f;
          coef[threadIdx.x][k][1] = ok ? ws * vy : 0.f;
          coef[threadIdx.x][k][2] = ok ? ws * vz : 0.f;
        }
      }
      __syncthreads();
      for (int j = 0; j < mc; ++j) {
        const int m = m0 + j;
#pragma unroll
        for (int i = 0; i < kOut; ++i) {
          const int n = n0 + i * kThreads + threadIdx.x;
          if (n >= m && n < nt) {
            const int lag = n - m;
            float a = 0.f;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const float* h = p.H + (size_t)node[j][k] * row + (size_t)lag * 3;
              a = fmaf(coef[j][k][0], __ldg(h), a);
              a = fmaf(coef[j][k][1], __ldg(h + 1), a);
              a = fmaf(coef[j][k][2], __ldg(h + 2), a);
            }
            acc[i] += a;
          }
        }
      }
    }
#pragma unroll
    for (int i = 0; i < kOut; ++i) {
      const int n = n0 + i * kThreads + threadIdx.x;
      if (n < nt) p.out[(size_t)c * nt + n] = acc[i];
    }
  }
}

// a12: i_track[n] = sum over the track's carriers in carrier order (fixed order: deterministic)
__global__ void __launch_bounds__(256) k_track_sum(const float* __restrict__ cur, const int64_t* __restrict__ track_off,
                                                   float* __restrict__ out, int nt) {
  const int64_t t = blockIdx.x;
  const int64_t c0 = track_off[t], c1 = track_off[t + 1];
  for (int n = threadIdx.x; n < nt; n += blockDim.x) {
    float s = 0.f;
    for (int64_t c = c0; c < c1; ++c) s += cur[(size_t)c * nt + n];
    out[(size_t)t * nt + n] = s;
  }
}

__global__ void k_nodes(int64_t n_steps, const float* __restrict__ pos, int32_t* __restrict__ n0, int32_t* __restrict__ n1,
                        float* __restrict__ fr, int nx, int ny, int nz, float invx, float invy, float invz) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n_steps) return;
  const NodeFrac nf = locate(pos[3 * s], pos[3 * s + 1], pos[3 * s + 2], nx, ny, nz, invx, invy, invz);
  for (int a = 0; a < 3; ++a) { n0[3 * s + a] = nf.i0[a]; n1[3 * s + a] = nf.i1[a]; fr[3 * s + a] = nf.f[a]; }
}

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

}  // namespace

extern "C" int wt_conv_workspace_bytes(const wt_geometry* g, int64_t n_tracks, int64_t n_carriers, int per_track,
                                       size_t* bytes) {
  if (!wt_valid(g) || !bytes || n_tracks < 0 || n_carriers < 0) { wt_set_error("wt_conv_workspace_bytes: bad argument"); return WT_EINVAL; }
  *bytes = per_track ? align_up((size_t)n_carriers * g->nt * sizeof(float)) : 0;
  return WT_OK;
}

extern "C" int wt_convolve_currents(const wt_geometry* g, const float* H_dev, int64_t n_tracks,
                                    const int64_t* track_carrier_offsets_dev, int64_t n_carriers,
                                    const int64_t* carrier_step_offsets_dev, const float* pos_dev, const float* vel_dev,
                                    const float* charge_dev, int per_track, float* out_dev, void* workspace_dev,
                                    size_t workspace_bytes, void* cuda_stream) {
  if (!wt_valid(g)) { wt_set_error("wt_convolve_currents: bad handle"); return WT_EINVAL; }
  const int64_t rows = per_track ? n_tracks : n_carriers;
  if (!H_dev || !carrier_step_offsets_dev || (!charge_dev && n_carriers > 0) || (!out_dev && rows > 0) || !cuda_stream ||
      n_carriers < 0 || n_tracks < 0 || (per_track && !track_carrier_offsets_dev)) {
    wt_set_error("wt_convolve_currents: null argument, negative count or NULL (default) stream"); return WT_EINVAL;
  }
  if (n_carriers > 0x7fffffffLL || n_tracks > 0x7fffffffLL) { wt_set_error("wt_convolve_currents: more than 2^31-1 carriers or tracks in one call"); return WT_EINVAL; }
  if ((size_t)g->nx * g->ny * g->nz > 0xffffffffull) { wt_set_error("wt_convolve_currents: grid too large"); return WT_EINVAL; }
  size_t need = 0;
  wt_conv_workspace_bytes(g, n_tracks, n_carriers, per_track, &need);
  if (need > 0 && (!workspace_dev || workspace_bytes < need)) {
    wt_set_error("wt_convolve_currents: workspace too small, need " + std::to_string(need)); return WT_ENOMEM;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  ConvParams p;
  p.H = H_dev; p.carrier_off = carrier_step_offsets_dev; p.pos = pos_dev; p.vel = vel_dev; p.charge = charge_dev;
  p.out = per_track ? (float*)workspace_dev : out_dev;
  p.nx = g->nx; p.ny = g->ny; p.nz = g->nz; p.nt = g->nt;
  p.invx = (float)((double)g->nx / g->lx); p.invy = (float)((double)g->ny / g->ly); p.invz = (float)((double)g->nz / g->lz);
  p.dt_over_vw = (float)(g->dt / g->v_w);
  if (n_carriers > 0) ++g_wt_launches;
  if (n_carriers > 0) k_conv_carrier<<<(unsigned)n_carriers, kThreads, 0, st>>>(p);
  if (per_track && n_tracks > 0) ++g_wt_launches;
  if (per_track && n_tracks > 0)
    k_track_sum<<<(unsigned)n_tracks, 256, 0, st>>>((const float*)workspace_dev, track_carrier_offsets_dev, out_dev, g->nt);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { wt_set_error(std::string("wt_convolve_currents: ") + cudaGetErrorString(e)); return WT_ECUDA; }
  wt_set_error("");
  return WT_OK;
}

extern "C" int wt_trajectory_nodes(const wt_geometry* g, int64_t n_steps, const float* pos_dev, int32_t* node0_dev,
                                   int32_t* node1_dev, float* frac_dev, void* cuda_stream) {
  if (!wt_valid(g) || n_steps < 0 || !cuda_stream || (n_steps > 0 && (!pos_dev || !node0_dev || !node1_dev || !frac_dev))) {
    wt_set_error("wt_trajectory_nodes: bad argument"); return WT_EINVAL;
  }
  if (n_steps > 0) ++g_wt_launches;
  if (n_steps > 0)
    k_nodes<<<(unsigned)((n_steps + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
        n_steps, pos_dev, node0_dev, node1_dev, frac_dev, g->nx, g->ny, g->nz, (float)((double)g->nx / g->lx),
        (float)((double)g->ny / g->ly), (float)((double)g->nz / g->lz));
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { wt_set_error(std::string("wt_trajectory_nodes: ") + cudaGetErrorString(e)); return WT_ECUDA; }
  wt_set_error("");
  return WT_OK;
}
