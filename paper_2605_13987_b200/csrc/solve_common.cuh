// Device-side descriptors shared by the kernels of wt_solve_H (solve.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace wt {

constexpr int kMaxLayers = 8;
constexpr int kStageSlots = 8;   // TB: output steps buffered before a table write (96-byte runs)

struct GridDev {
  int nx, ny, nz, y2, nt, ty, n_tiles;   // generic k_spectral: ty lines per CTA, n_tiles = nx * (y2/ty)
  double inv_n;
  const int* step;                        // device counter: index n of the output step being produced
};

struct GeomDev {
  // static tables
  const uint8_t* sig_id;     // [z][x][y]  0 = diamond, j+1 = column j     (generic plane kernel)
  const uint8_t* sig_t;      // [z][y][x]                                   (size-specialised plane kernel)
  const float* sdt;          // [256]  s * dt_int of id
  const float* gt;           // [kx][dz][ky] mixed-space fundamental solution
  const float* gzt;          //              and its -d/dz
  const double* ainv;        // [B][B]
  const double* pad_pot;     // [B]
  const int* pad_y;          // [B]
  // pads grouped by (layer, x): group k covers grp_pad[grp_off[k] .. grp_off[k+1])
  const int* grp_x;          // [G]
  const int* grp_layer;      // [G]
  const int* grp_off;        // [G+1]
  const int* grp_pad;        // [B] pad indices in group order
  const int* layer_goff;     // [L+1] groups of layer l = [layer_goff[l], layer_goff[l+1])
  const double* kxd; const double* kyd; const double* kzd;    // wavenumbers (0 at the removed Nyquist index)
  const float* kxf; const float* kyf; const float* kzf;
  const float2* twx; const float2* twy; const float2* twz;    // e^{-2 pi i k/n}
  const double2* twxd; const double2* twyd; const double2* twzd;
  // state
  double2* rhat; double2* rhat_prev;   // [kx][kz][ky]   charge spectrum r = rho/eps (fp64)
  float2* m0; float2* m1;              // step pipeline: (V~_rho | D~), (E~z_rho | J~z)   [kx][z][ky]
  float2* e0; float2* e1;              // emit pipeline
  double2* pl; double2* pl_e;          // [L][kx][ky]  V~_rho at the pad layers (fp64), step / emit pipeline
  double* rhs; double* q;              // [B]
  float2* qh;                          // [L][kx][ky] spectrum of the boundary charges
  float* stage;                        // [TB][3][z][..] staging of H for the time-innermost table write
  float* H;
  int layers[kMaxLayers];
  int B, L, G, n_sub;
  float inv_dt;
};

__device__ __forceinline__ double2 dmul(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

}  // namespace wt
