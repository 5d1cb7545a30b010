// wt_convolve_currents / wt_trajectory_nodes: steps a9-a12 of the hot path (Eq. 1.1).
//
// PAPER.md:35-39 (Eq. 1.1), :74 ("for each charge carrier, the induced signal is computed as
// described in Equation 1.1"), :99 (one carrier per CUDA thread, H through texture interpolation).
// Two kernels compute the same sums:
//   k_conv_systolic (nt <= 1024)  one CTA per group of consecutive carriers; lanes own FLOATS of the
//       time-innermost rows (16-byte aligned, fully coalesced 128-bit loads) and the partial sums
//       travel across the lanes by warp shuffles as the step index advances (see the kernel);
//   k_conv_carrier (any nt)       one CTA per carrier, threads own output times n.
// Trilinear weights in full fp32 (R23).  Per-track sums are formed in carrier order from partial
// rows in a second pass (R25: fixed order, no float atomics).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <mutex>
#include <string>

#include "geometry.h"
#include "locate.cuh"

namespace {
using wt::NodeFrac;
using wt::locate;

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

// ------------------------------------------------------------------------------------------------
// k_conv_systolic: Eq. 1.1 with the table rows read where they lie.
//
// A node row is F = 3 nt floats, float f = 3 lag + component.  Step m, corner k adds
//   c[m][k][f % 3] * row_k[f]   to the partial sum   S[f + 3 m],       i(n) = S[3n] + S[3n+1] + S[3n+2].
// Warp w owns the floats [384 w, 384 w + 384) of every row: lane t holds f = 384 w + 128 j + 4 t + i
// (j < 3, i < 4), i.e. three 128-bit loads per corner that are 16-byte aligned for every step and
// cover 512 contiguous bytes per instruction.  The twelve partial sums of a lane belong to S[f + 3 m]:
// when m advances they move down by three floats, i.e. one register rotation plus three shuffles per
// 128-float group; sums that leave the warp's range at the bottom are complete (for this warp) and go
// to the warp's own row P_w in shared memory, each element written once per carrier, so the result
// does not depend on scheduling (R25).  Component of (j, i) = (t + 2 j + i) % 3: the three weights of
// a corner are rotated by t % 3 once per corner with selects.
// One CTA handles `gc` consecutive carriers; with per_track the rows of carriers of one track are
// summed in P (carrier order) and written as one partial row at the index of the segment's first carrier.
// grid = ceil(n_carriers / gc), block = 32 * ceil(nt / 128) <= 256 (cached kernel: 384, as many warps as have a partial row in 220 KB),
// dynamic smem = step table (32 steps of 128 bytes; cached kernel 128 steps of 328 bytes) + the partial rows, warp w's being
// the F - 384 w floats it can reach (55 KB instead of 98 KB at nt = 1024, which goes to L1).
// ------------------------------------------------------------------------------------------------
constexpr int kStepChunk = 32;        // steps per step table: plain kernel (carriers of a few dozen steps)
constexpr int kCachedThreads = 384;   // cached kernel: twelve warps share the eight lag blocks of nt = 1024 (162 registers, one CTA per SM)
constexpr int kStepChunkCached = 128;  // cached kernel (nt >= 1024, hundreds of steps: fewer table builds, during which seven warps wait)

// shared memory of the systolic kernel: bytes per step of the step table, and the float offset of warp w's partial row
// (rows of F - 384 u floats, u < w, lie before it)
constexpr int kStepBytesPlain = 8 * sizeof(float4);                                         // 8 (node, w) pairs + velocity + (unused) key
constexpr int kStepBytesCached = 3 * 24 * sizeof(float) + 8 * sizeof(unsigned) + sizeof(unsigned long long);
__host__ __device__ constexpr int rows_offset(int w, int F) { return w * F - 192 * w * (w - 1); }

struct SysParams {
  ConvParams c;
  const int64_t* track_off;   // [n_tracks + 1] (per_track) or NULL
  int64_t n_tracks, n_carriers;
  int gc, stride, per_track;   // a CTA handles carriers base + s, base + s + stride, ... (gc of them)
};

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// CACHE: the 8 x 12 floats a lane owns of the current cell's rows stay in registers while the carrier stays in the cell
// (a carrier of configs[2] / [4] spends 2-4 steps per cell: those steps are pure FMA + shuffle, no row is read again); the
// step table then holds, per step, the 24 products (w_k * scale) * v_c once for each of the three rotations of the components a
// lane can need (six 128-bit shared loads per step instead of 24 multiplies and six selects), the eight nodes and a cell key.
// FULL: nt is a multiple of 128, so every lane of every warp owns three whole 16-byte groups of a row and the row loads need no
// predicates (all BASELINE configs).
template <bool CACHE, bool FULL>
__global__ void __launch_bounds__(CACHE ? kCachedThreads : 256, CACHE ? 1 : 2) k_conv_systolic(SysParams sp) {
  constexpr int CH = CACHE ? kStepChunkCached : kStepChunk;
  constexpr int kStepBytes = CACHE ? kStepBytesCached : kStepBytesPlain;
  const ConvParams& p = sp.c;
  const int nt = p.nt, F = 3 * nt;
  const int tid = threadIdx.x, w = tid >> 5, t = tid & 31, nw = blockDim.x >> 5;     // nw warps
  const int nb = (nt + 127) >> 7;                                                        // nb lag blocks of 128 lags (= nw unless BAL)
  extern __shared__ __align__(16) unsigned char smraw[];
  // BAL (cached kernel): the (lag block, step) pairs of a step table are dealt out evenly to the warps, see below; a warp then
  // holds sums of any block and its partial row is all F floats.  Otherwise warp w owns block w and only ever holds sums
  // S[g], g >= 384 w: its row is the F - 384 w floats [384 w, F).
  constexpr bool BAL = CACHE;
  float* P = reinterpret_cast<float*>(smraw + CH * kStepBytes);
  float* Pw = BAL ? P + (size_t)w * F : P + rows_offset(w, F) - 384 * w;    // Pw[g]
  const int p_floats = BAL ? nw * F : rows_offset(nw, F);
  __shared__ int64_t s_track;
  __shared__ unsigned s_cmask[kStepChunkCached / 32];   // cached kernel: where the carrier changes cell inside the step table
  // step table: per step eight (node, w * scale) pairs, the velocity and (CACHE) the cell key
  float2* tabc = reinterpret_cast<float2*>(smraw);                                // [CH][8]
  float4* tabv = reinterpret_cast<float4*>(smraw + CH * 8 * sizeof(float2));          // [CH]
  unsigned long long* keys = reinterpret_cast<unsigned long long*>(smraw + CH * (8 * sizeof(float2) + sizeof(float4)));   // [CH] (plain kernel: unused)
  // cached kernel: per step the 24 products (w_k * scale) * v_c for each of the three rotations of the components a lane can
  // need (lane t multiplies float f of a row by component (t + f) % 3), the eight nodes and the cell key
  float4* tabq = reinterpret_cast<float4*>(smraw);                                                         // [CH][3][6]
  unsigned* tabn = reinterpret_cast<unsigned*>(smraw + CH * 3 * 24 * sizeof(float));                       // [CH][8]
  if constexpr (CACHE) keys = reinterpret_cast<unsigned long long*>(smraw + CH * (3 * 24 * sizeof(float) + 8 * sizeof(unsigned)));

  const int r = t % 3;
  const bool r0 = (r == 0), r1 = (r == 1);

  // carriers of this CTA: cb, cb + S, cb + 2 S, ... (gc of them, inside one super-group of gc * S carriers):
  // the S CTAs of a super-group work on S adjacent carriers at any time, whose rows largely coincide (L2 reuse)
  const int S = sp.stride;
  const int64_t sgb = (int64_t)(blockIdx.x / S) * sp.gc * S;
  const int64_t cb = sgb + blockIdx.x % S, ce = min(sp.n_carriers, sgb + (int64_t)sp.gc * S);
  if (cb >= ce) return;
  // track of the first carrier: largest tr with track_off[tr] <= cb
  int64_t tr = 0, c_next = 0x7fffffffffffffffLL, seg = cb;
  if (sp.per_track) {
    if (tid == 0) {
      int64_t lo = 0, hi = sp.n_tracks;            // invariant: track_off[lo] <= cb (track_off[0] may exceed cb: handled below)
      while (lo < hi) { const int64_t mid = (lo + hi + 1) >> 1; if (sp.track_off[mid] <= cb) lo = mid; else hi = mid - 1; }
      s_track = lo;
    }
    __syncthreads();
    tr = s_track;
    if (tr >= sp.n_tracks) return;                 // carriers past the last track belong to no row
    c_next = sp.track_off[tr + 1];
    seg = max(cb, sp.track_off[tr]);               // first carrier index that can open a segment
  }
  for (int i = tid; i < p_floats; i += blockDim.x) P[i] = 0.f;
  __syncthreads();
  bool opened = false;

  // writes i(n) = sum_w S_w[3n..3n+2] to the output row and clears P
  auto flush_row = [&](float* __restrict__ row) {
    __syncthreads();
    for (int n = tid; n < nt; n += blockDim.x) {
      float s = 0.f;
      for (int ww = 0; BAL ? ww < nw : 128 * ww <= n; ++ww) {   // (!BAL: warp ww holds S[g] for g >= 384 ww only; 128 ww <= n < nt keeps ww < nw)
        const float* q = (BAL ? P + (size_t)ww * F : P + rows_offset(ww, F) - 384 * ww) + 3 * n;
        s += (q[0] + q[1]) + q[2];
      }
      row[n] = s;
    }
    __syncthreads();
    for (int i = tid; i < p_floats; i += blockDim.x) P[i] = 0.f;
    __syncthreads();
  };

  for (int64_t c = cb; c < ce; c += S) {
    if (c < seg) continue;                         // (carriers before the first track belong to no row)
    if (sp.per_track && c >= c_next) {             // the track changes inside the group
      if (opened) flush_row(p.out + (size_t)seg * nt);
      opened = false;
      while (tr < sp.n_tracks && c >= sp.track_off[tr + 1]) ++tr;
      if (tr >= sp.n_tracks) return;
      c_next = sp.track_off[tr + 1];
    }
    if (!opened) { opened = true; seg = c; }       // partial rows live at the index of the segment's first carrier
    const int64_t s0 = p.carrier_off[c];
    const int M = (int)min((int64_t)nt, p.carrier_off[c + 1] - s0);   // steps m >= nt are ignored (R26)
    const float scale = -p.charge[c] * p.dt_over_vw;
    float A[3][4];
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int i = 0; i < 4; ++i) A[j][i] = 0.f;

    // m -> m + 1: the sums move down by three floats; the three lowest of the warp are complete
    // (lane 0 reads the three sums it will complete at the top of the step, pre(), and writes them back in shift(): the shared
    // load is then not waited for behind the step's 96 FMA)
    float pq[3] = {0.f, 0.f, 0.f};
    auto pre = [&](int u, int m) {
      const int gq = 384 * u + 3 * m;
      if (t == 0 && gq < F) { pq[0] = Pw[gq]; pq[1] = Pw[gq + 1]; pq[2] = Pw[gq + 2]; }     // F % 3 == 0
    };
    auto shift = [&](int u, int m) {
      {
        const int gq = 384 * u + 3 * m;
        if (t == 0 && gq < F) { Pw[gq] = pq[0] + A[0][0]; Pw[gq + 1] = pq[1] + A[0][1]; Pw[gq + 2] = pq[2] + A[0][2]; }
      }
      float sh[3][3];
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          const float up = (j < 2) ? A[j + 1][i] : 0.f;
          sh[j][i] = __shfl_sync(0xffffffffu, t == 0 ? up : A[j][i], (t + 1) & 31);
        }
#pragma unroll
      for (int j = 0; j < 3; ++j) { A[j][0] = A[j][3]; A[j][1] = sh[j][0]; A[j][2] = sh[j][1]; A[j][3] = sh[j][2]; }
    };
    // one (step, corner) entry e = (., c_x, c_y, c_z) applied to the lane's twelve floats of the corner's row
    auto fma12q = [&](float (&D)[3][4], const float q0, const float q1, const float q2, const float4 h0, const float4 h1, const float4 h2) {
      D[0][0] = fmaf(q0, h0.x, D[0][0]); D[0][1] = fmaf(q1, h0.y, D[0][1]); D[0][2] = fmaf(q2, h0.z, D[0][2]); D[0][3] = fmaf(q0, h0.w, D[0][3]);
      D[1][0] = fmaf(q2, h1.x, D[1][0]); D[1][1] = fmaf(q0, h1.y, D[1][1]); D[1][2] = fmaf(q1, h1.z, D[1][2]); D[1][3] = fmaf(q2, h1.w, D[1][3]);
      D[2][0] = fmaf(q1, h2.x, D[2][0]); D[2][1] = fmaf(q2, h2.y, D[2][1]); D[2][2] = fmaf(q0, h2.z, D[2][2]); D[2][3] = fmaf(q1, h2.w, D[2][3]);
    };
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 HC[CACHE ? 8 : 1][3];
    unsigned long long cell_key = ~0ULL;             // (per carrier: the first step always loads)

    {
      for (int m0 = 0; m0 < M; m0 += CH) {
        const int mc = min(CH, M - m0);
        __syncthreads();
        for (int js = tid; js < mc; js += blockDim.x) {
          const int64_t s = s0 + m0 + js;
          const float vx = p.vel[3 * s], vy = p.vel[3 * s + 1], vz = p.vel[3 * s + 2];
          const NodeFrac nf = locate(p.pos[3 * s], p.pos[3 * s + 1], p.pos[3 * s + 2], p.nx, p.ny, p.nz, p.invx, p.invy, p.invz);
          const bool ok = nf.ok && isfinite(vx) && isfinite(vy) && isfinite(vz);
          unsigned key_hi = 0;
          unsigned long long key = 0;
          float wsk[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const int cx = k >> 2, cy = (k >> 1) & 1, cz = k & 1;
            const float wgt = (cx ? nf.f[0] : 1.f - nf.f[0]) * (cy ? nf.f[1] : 1.f - nf.f[1]) * (cz ? nf.f[2] : 1.f - nf.f[2]);
            const int ix = cx ? nf.i1[0] : nf.i0[0], iy = cy ? nf.i1[1] : nf.i0[1], iz = cz ? nf.i1[2] : nf.i0[2];
            const unsigned node = ok ? (unsigned)((ix * p.ny + iy) * p.nz + iz) : 0u;
            const float ws = wgt * scale;            // a non-finite step contributes nothing (0, not 0 * inf)
            wsk[k] = ok ? ws : 0.f;
            if constexpr (CACHE) {
              tabn[js * 8 + k] = node;
              if (k == 0) key_hi = node;
              if (k == 7) key = ((unsigned long long)key_hi << 32) | node;   // corners 0 and 7 identify the cell (a skipped step has both 0: never a real cell)
            } else {
              tabc[js * 8 + k] = make_float2(__uint_as_float(node), wsk[k]);
            }
          }
          if constexpr (CACHE) {
            keys[js] = key;
            // bit j of the change mask: step j + 1 of this table opens another cell than step j (taken as set across the
            // 32-step words, where the neighbour's key is not at hand: the prefetch it triggers then asks for rows already near)
            const unsigned act = __activemask();
            const unsigned long long nk = __shfl_down_sync(act, key, 1);
            const unsigned mw = __ballot_sync(act, (js + 1 < mc) && (t == 31 || nk != key));
            if (t == 0) s_cmask[js >> 5] = mw;
            const float v3[3] = {ok ? vx : 0.f, ok ? vy : 0.f, ok ? vz : 0.f};
#pragma unroll
            for (int rot = 0; rot < 3; ++rot) {
              float q[24];
#pragma unroll
              for (int k = 0; k < 8; ++k)
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) q[3 * k + cc] = wsk[k] * v3[(rot + cc) % 3];
#pragma unroll
              for (int i = 0; i < 6; ++i) tabq[(js * 3 + rot) * 6 + i] = make_float4(q[4 * i], q[4 * i + 1], q[4 * i + 2], q[4 * i + 3]);
            }
          } else {
            tabv[js] = ok ? make_float4(vx, vy, vz, 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
          }
        }
        __syncthreads();
        // Lag block u (floats [384 u, 384 u + 384) of the rows) has outputs below nt for the steps m < nt - 128 u only (the causal
        // triangle): with one block per warp, warp nw - 1 is done after 128 steps, the next after 256, ... and their schedulers
        // idle.  BAL: the live (block, step) pairs of this table, block-major, are cut into nw equal runs, one per warp; a warp
        // starts each of its (at most three) pieces with empty sums and leaves them in its own row at the end of the piece, so
        // the result depends on nt, M and nw only (R25).  The CTA has more warps than blocks (twelve for the eight blocks of nt = 1024).
        int lo = 0, hi = mc;
        if constexpr (BAL) {
          int total = 0;
          for (int u = 0; u < nb; ++u) total += max(0, min(mc, nt - 128 * u - m0));
          const int per = (total + nw - 1) / nw;
          lo = w * per; hi = min(total, lo + per);
        }
        int base = 0;
        for (int u = BAL ? 0 : w; u < (BAL ? nb : w + 1); ++u) {
        const int len = BAL ? max(0, min(mc, nt - 128 * u - m0)) : mc;
        const int ja = BAL ? max(lo, base) - base : 0, jb = BAL ? min(hi, base + len) - base : mc;
        base += len;
        if (ja >= jb) continue;
        const int f0 = 384 * u + 4 * t;
        const bool v0 = FULL || f0 < F, v1 = FULL || f0 + 128 < F, v2 = FULL || f0 + 256 < F;       // F % 4 == 0: whole 16-byte groups
        if constexpr (BAL) {
#pragma unroll
          for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int i = 0; i < 4; ++i) A[j][i] = 0.f;
          cell_key = ~0ULL;
        }
        int jm = ja;
        for (; jm < jb; ++jm) {
          const int m = m0 + jm;
          if (128 * u + m >= nt) break;              // every output of this block is past nt from here on (warp uniform)
          pre(u, m);
          if constexpr (CACHE) {
            const unsigned long long key = keys[jm];
            if (key != cell_key) {                   // (warp uniform)
              cell_key = key;
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const float* __restrict__ src = p.H + (size_t)tabn[jm * 8 + k] * F + f0;
                HC[k][0] = v0 ? ldg4(src) : z4; HC[k][1] = v1 ? ldg4(src + 128) : z4; HC[k][2] = v2 ? ldg4(src + 256) : z4;
              }
              {
                // the next cell of this table is asked into L2 now: its rows arrive while the steps inside this cell are
                // summed (tables beyond L2: +10 % at configs[4]).  A warp's share of 8 rows is 8 x 12 lines of 128 bytes:
                // three per lane.
                const unsigned word = s_cmask[jm >> 5] >> (jm & 31);
                const int jn = jm + __ffs(word);
                if (word != 0 && jn < mc) {
#pragma unroll
                  for (int i = 0; i < 3; ++i) {
                    const int idx = t + 32 * i, k = idx / 12, l = idx - 12 * k;
                    const int fo = 384 * u + 32 * l;
                    const float* a = p.H + (size_t)tabn[jn * 8 + k] * F + fo;
                    if (FULL || fo < F) asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
                  }
                }
              }
            }
            const float4* tq = tabq + (jm * 3 + r) * 6;
            float q[24];
#pragma unroll
            for (int i = 0; i < 6; ++i) { const float4 e = tq[i]; q[4 * i] = e.x; q[4 * i + 1] = e.y; q[4 * i + 2] = e.z; q[4 * i + 3] = e.w; }
#pragma unroll
            for (int k = 0; k < 8; ++k) fma12q(A, q[3 * k], q[3 * k + 1], q[3 * k + 2], HC[k][0], HC[k][1], HC[k][2]);
          } else {
            const float4 vv = tabv[jm];
            const float q0 = r0 ? vv.x : (r1 ? vv.y : vv.z);      // velocity component (t + x) % 3, x = 0, 1, 2
            const float q1 = r0 ? vv.y : (r1 ? vv.z : vv.x);
            const float q2 = r0 ? vv.z : (r1 ? vv.x : vv.y);
            const float4* tc4 = reinterpret_cast<const float4*>(tabc + jm * 8);
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              const float4 e2 = tc4[kk];             // (node, w * scale) of corners 2 kk and 2 kk + 1
              {
                const float* __restrict__ src = p.H + (size_t)__float_as_uint(e2.x) * F + f0;
                const float4 h0 = v0 ? ldg4(src) : z4, h1 = v1 ? ldg4(src + 128) : z4, h2 = v2 ? ldg4(src + 256) : z4;
                fma12q(A, e2.y * q0, e2.y * q1, e2.y * q2, h0, h1, h2);
              }
              {
                const float* __restrict__ src = p.H + (size_t)__float_as_uint(e2.z) * F + f0;
                const float4 h0 = v0 ? ldg4(src) : z4, h1 = v1 ? ldg4(src + 128) : z4, h2 = v2 ? ldg4(src + 256) : z4;
                fma12q(A, e2.w * q0, e2.w * q1, e2.w * q2, h0, h1, h2);
              }
            }
          }
          shift(u, m);
        }
        if constexpr (BAL) {
          // after the steps [m0 + ja, m0 + jm) lane (j, i) holds its share of S[f + 3 (m0 + jm)]
          __syncwarp();
#pragma unroll
          for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int gq = f0 + 128 * j + i + 3 * (m0 + jm);
              if (f0 + 128 * j < F && gq < F) Pw[gq] += A[j][i];
            }
          __syncwarp();
        }
        }
      }
    }
    if constexpr (!BAL) {
      // after M steps lane (j, i) holds S[f + 3 M]
      const int f0 = 384 * w + 4 * t;
      __syncwarp();
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int gq = f0 + 128 * j + i + 3 * M;
          if (f0 + 128 * j < F && gq < F) Pw[gq] += A[j][i];   // (a warp that left the loop early holds outputs >= nt only)
        }
      __syncwarp();
    }
    if (!sp.per_track) flush_row(p.out + (size_t)c * nt);
  }
  if (sp.per_track && opened) flush_row(p.out + (size_t)seg * nt);
}

// a12: i_track[n] = sum of the partial rows of the track in carrier order (fixed order: deterministic).
// A CTA of the convolution kernel handles the carriers base + s + i * stride (i < gc) of a super-group of
// gc * stride carriers and leaves one partial row per track segment at the index of the segment's first
// carrier; gc = 1: one row per carrier.
__global__ void __launch_bounds__(256) k_track_sum(const float* __restrict__ cur, const int64_t* __restrict__ track_off,
                                                   float* __restrict__ out, int nt, int gc, int stride) {
  const int64_t t = blockIdx.x;
  const int64_t c0 = track_off[t], c1 = track_off[t + 1], sg = (int64_t)gc * stride;
  __shared__ int64_t rows[256];
  __shared__ int n_rows;
  __shared__ int64_t c_resume;
  for (int nb = 0; nb < nt; nb += 4 * 256) {
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    int64_t c = c0;
    while (c < c1) {                                 // (uniform: c comes from shared memory)
      __syncthreads();
      if (threadIdx.x == 0) {
        // segment starts: carriers whose predecessor in their CTA (c - stride) lies outside the track or the super-group
        int k = 0;
        while (c < c1 && k < 256) {
          const int64_t base = c / sg * sg;
          if (c - stride < c0 || c - stride < base) rows[k++] = c++;
          else c = base + sg;
        }
        n_rows = k; c_resume = c;
      }
      __syncthreads();
      for (int r = 0; r < n_rows; ++r) {
        const float* __restrict__ row = cur + (size_t)rows[r] * nt + nb + threadIdx.x;
#pragma unroll
        for (int i = 0; i < 4; ++i)
          if (nb + i * 256 + (int)threadIdx.x < nt) acc[i] += row[i * 256];
      }
      c = c_resume;
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
      if (nb + i * 256 + (int)threadIdx.x < nt) out[(size_t)t * nt + nb + i * 256 + threadIdx.x] = acc[i];
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

bool env_flag(const char* name) {
  const char* v = std::getenv(name);
  return v && v[0] && v[0] != '0';
}

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
  if (((uintptr_t)H_dev) % 16 != 0) { wt_set_error("wt_convolve_currents: H table not 16-byte aligned (rows are read with 128-bit loads)"); return WT_EINVAL; }
  if (workspace_dev && ((uintptr_t)workspace_dev) % 256 != 0) { wt_set_error("wt_convolve_currents: workspace not 256-byte aligned"); return WT_EINVAL; }
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
  // kernel choice: the systolic kernel for nt <= 1024 (its per-warp rows fit in shared memory), else one CTA per carrier
  const bool force_v1 = env_flag("WTIDE_CONV_V1");   // (read per call, like the switches of wt_solve_H)
  const int nw = (g->nt + 127) / 128;
  int gc = 1, stride = 1;
  if (n_carriers > 0 && nw <= 8 && !force_v1) {
    if (per_track && n_carriers >= 148 * 8 * 8) { gc = 8; stride = 32; }   // carriers per CTA: amortises the row combine
    SysParams sp;
    sp.c = p; sp.track_off = per_track ? track_carrier_offsets_dev : nullptr;
    sp.n_tracks = n_tracks; sp.n_carriers = n_carriers; sp.gc = gc; sp.stride = stride; sp.per_track = per_track ? 1 : 0;
    // rows cached in registers across the steps a carrier spends in one cell: pays when carriers take several steps per cell
    // (fine time grids: nt >= 1024 in the BASELINE configs); WTIDE_CONV_CACHE=0/1 forces either kernel (both parity-tested)
    bool cache = g->nt >= 1024;
    if (const char* ev = std::getenv("WTIDE_CONV_CACHE")) cache = ev[0] == '1';
    const bool full = g->nt % 128 == 0;
    auto fn = cache ? (full ? k_conv_systolic<true, true> : k_conv_systolic<true, false>) : (full ? k_conv_systolic<false, true> : k_conv_systolic<false, false>);
    // cached kernel: warps beyond the nw lag blocks (its work is dealt out per (block, step)); each needs a full partial row
    int warps = nw;
    if (cache) {
      warps = kCachedThreads / 32;
      const size_t row = (size_t)3 * g->nt * sizeof(float), room = 220 * 1024 - (size_t)kStepChunkCached * kStepBytesCached;
      warps = (int)std::max<size_t>(1, std::min<size_t>(warps, room / row));
    }
    const size_t smem = (cache ? (size_t)kStepChunkCached * kStepBytesCached : (size_t)kStepChunk * kStepBytesPlain) +
                        (size_t)(cache ? warps * 3 * g->nt : rows_offset(nw, 3 * g->nt)) * sizeof(float);
    cudaError_t ea = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (ea != cudaSuccess) { wt_set_error(std::string("wt_convolve_currents: ") + cudaGetErrorString(ea)); return WT_ECUDA; }
    ++g_wt_launches;
    const int64_t sg = (int64_t)gc * stride;
    fn<<<(unsigned)((n_carriers + sg - 1) / sg * stride), 32 * warps, smem, st>>>(sp);
  } else if (n_carriers > 0) {
    ++g_wt_launches;
    k_conv_carrier<<<(unsigned)n_carriers, kThreads, 0, st>>>(p);
  }
  if (per_track && n_tracks > 0) {
    ++g_wt_launches;
    k_track_sum<<<(unsigned)n_tracks, 256, 0, st>>>((const float*)workspace_dev, track_carrier_offsets_dev, out_dev, g->nt, gc, stride);
  }
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

// ---- Eq. 1.1 per track without any allocation ------------------------------------------------------------------
// For callers that cannot call cudaMalloc (tight serving loops, harnesses that forbid it): the per-carrier rows that
// wt_convolve_currents(per_track = 1) keeps in a caller workspace live in a file-scope device array instead.  Every GPU
// that loads the library holds WT_NOALLOC_MAX_FLOATS * 4 bytes (4 MiB) of it until exit.  In host code the array's name is
// a host-side stand-in, not a device address: its device address is looked up once per device (with that device current)
// by cudaGetSymbolAddress and handed to the same kernels the workspace form launches.
static __device__ __align__(256) float g_noalloc_rows[WT_NOALLOC_MAX_FLOATS];

namespace {
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
float* g_noalloc_ptr[kNoAllocMaxDevices];   // device address of g_noalloc_rows on device d (NULL: not looked up yet)
}  // namespace

extern "C" int wt_convolve_tracks_noalloc(const wt_geometry* g, const float* H_dev, int64_t n_tracks,
                                          const int64_t* track_carrier_offsets_dev, int64_t n_carriers,
                                          const int64_t* carrier_step_offsets_dev, const float* pos_dev, const float* vel_dev,
                                          const float* charge_dev, float* out_dev, void* cuda_stream) {
  if (!wt_valid(g)) { wt_set_error("wt_convolve_tracks_noalloc: bad handle"); return WT_EINVAL; }
  if (n_tracks < 0 || n_carriers < 0) { wt_set_error("wt_convolve_tracks_noalloc: negative count"); return WT_EINVAL; }
  if (n_carriers > (int64_t)WT_NOALLOC_MAX_FLOATS / g->nt) {
    wt_set_error("wt_convolve_tracks_noalloc: n_carriers * nt = " + std::to_string(n_carriers) + " * " + std::to_string(g->nt) +
                 " exceeds the built-in scratch of WT_NOALLOC_MAX_FLOATS = " + std::to_string((long long)WT_NOALLOC_MAX_FLOATS) +
                 " floats; split the batch or call wt_convolve_currents with a workspace");
    return WT_ENOMEM;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { wt_set_error(std::string("wt_convolve_tracks_noalloc: ") + cudaGetErrorString(e)); return WT_ECUDA; }
  if (dev < 0 || dev >= kNoAllocMaxDevices) { wt_set_error("wt_convolve_tracks_noalloc: device ordinal beyond 63"); return WT_EINVAL; }
  float* rows = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_noalloc_rows);
      if (e != cudaSuccess || !p) {
        wt_set_error(std::string("wt_convolve_tracks_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        return WT_ECUDA;
      }
      g_noalloc_ptr[dev] = (float*)p;
    }
    rows = g_noalloc_ptr[dev];
  }
  // The kernels write every row k_track_sum reads before it reads it (one row per carrier, or per segment of a carrier
  // group), so nothing in the array has to start at zero and what the last call left there is never read.
  const int rc = wt_convolve_currents(g, H_dev, n_tracks, track_carrier_offsets_dev, n_carriers, carrier_step_offsets_dev, pos_dev,
                                      vel_dev, charge_dev, 1, out_dev, rows, (size_t)WT_NOALLOC_MAX_FLOATS * sizeof(float), cuda_stream);
  return rc;
}
