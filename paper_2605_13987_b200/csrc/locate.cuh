// R24: the index arithmetic of the ABI (include/wtide.h), shared by Eq. 1.1 (conv.cu) and the transport kernels (next.cu).
#pragma once
#include <cuda_runtime.h>

namespace wt {

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

}  // namespace wt
