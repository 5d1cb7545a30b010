// Device-side descriptors shared by the kernels of wt_solve_H (solve.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace wt {

constexpr int kMaxLayers = 8;
constexpr int kStageSlots = 8;   // TB: output steps buffered before a table write (96-byte runs)
constexpr int kBatch = 8;        // geometries per launch: their descriptors travel as kernel parameters

struct GridDev {
  int nx, ny, nz, y2, nt, ty, n_tiles;   // generic k_spectral: ty lines per CTA, n_tiles = nx * (y2/ty)
  double inv_n;
  const int* step;                        // device counter: index n of the output step being produced
#ifdef WTIDE_DEBUG
  long long* stamps;                      // -DWTIDE_DEBUG builds with WTIDE_STAMPS=1: [16 ranks][16] clock stamps of the boundary kernel, else NULL
#endif
};

// One geometry of the lock-step batch.  Passed BY VALUE inside GeomBatch (kernel parameter space =
// constant bank): pointers and scalars cost neither a register nor a dependent global load.
// Pads are held in GROUP order (sorted by layer, then x, then y); "group" = pads of one (layer, x).
struct GeomDev {
  // static tables
  const uint8_t* sig_id;     // [z][x][y]  0 = diamond, j+1 = column j     (generic plane kernel)
  const uint8_t* sig_t;      // [z][y][x]                                   (size-specialised plane kernel)
  const float* sdt;          // [256]  s * dt_int of id
  const float* gt;           // [kx][dz][ky] mixed-space fundamental solution
  const float* gzt;          //              and its -d/dz
  const double* ainv;        // [B][Bs] in group order, row stride Bs = B rounded up to even (16-byte rows)
  const double* pad_pot;     // [B]
  const int* pad_y;          // [B]
  const int* grp_x;          // [G]
  const int* grp_layer;      // [G]
  const int* grp_off;        // [G+1] pads of group k = [grp_off[k], grp_off[k+1])
  const int* layer_goff;     // [L+1] groups of layer l = [layer_goff[l], layer_goff[l+1])
  const double* kxd; const double* kyd; const double* kzd;    // wavenumbers (0 at the removed Nyquist index)
  const float* kxf; const float* kyf; const float* kzf;
  const float2* twx; const float2* twy; const float2* twz;    // e^{-2 pi i k/n}
  const double2* twxd; const double2* twyd; const double2* twzd;
  // state
  double2* rhat; double2* rhat_prev;   // [kx][kz][ky]   charge spectrum r = rho/eps (fp64)
  float2* v0; float2* v1;              // z-line -> plane:  V~_rho, E~z_rho                      [kx][z][ky]
  float2* m0; float2* m1; float2* m2;  // plane -> z-line:  i kx J~x, i ky J~y, J~z              [kx][z][ky]
  float2* e0; float2* e1;              // emit pipeline (z-line -> plane)
  double2* pl; double2* pl_e;          // [L][kx][ky]  V~_rho at the pad layers (fp64), step / emit pipeline
  double* rhs; double* q;              // [B]
  float2* qh;                          // [L][kx][ky] spectrum of the boundary charges
  float* stage;                        // [TB][3][z][..] staging of H for the time-innermost table write
  float* H;
  int layers[kMaxLayers];
  int lgoff[kMaxLayers + 1];           // copy of layer_goff in the parameter space
  int B, Bs, L, G, n_sub;
  float inv_dt;
};

struct GeomBatch { GeomDev g[kBatch]; };

// Programmatic dependent launch (PDL): every kernel of wt_solve_H lets its successor start launching at
// once (its CTAs fill SMs as ours drain and run their prologue, which reads static tables only) and
// waits for the full completion of its predecessor before touching anything a kernel writes.
// Both are no-ops when the kernel was launched without the PDL attribute.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ double2 dmul(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

}  // namespace wt
