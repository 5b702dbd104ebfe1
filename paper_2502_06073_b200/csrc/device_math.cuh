// device_math.cuh — per-edge basis functions of the Allegro network on the device (fp32 unless noted).
// F1 envelope, F2 Bessel basis, F3 real spherical harmonics (PAPER.md:93 names only
// "e3nn", "l=2": the explicit forms are readings A1-A3).
#pragma once
#include <cuda_runtime.h>

namespace allegro {

// SiLU and its derivative with the fast reciprocal (MUFU.RCP, <= 2 ulp): the IEEE division costs ~10 more instructions
// per element and the MLP epilogues are issue-bound (profiles/r1_c_launches.md)
__device__ __forceinline__ float silu_f(float z) { return __fdividef(z, 1.0f + __expf(-z)); }
__device__ __forceinline__ float dsilu_f(float z) {
  float s = __fdividef(1.0f, 1.0f + __expf(-z));
  return s * (1.0f + z * (1.0f - s));
}

// Component-normalised real spherical harmonics, m = -l..l, polar axis z (F3).  Y has (lmax+1)^2 entries.
template <int LMAX>
__device__ __forceinline__ void sph_harm(float x, float y, float z, float* Y) {
  Y[0] = 1.0f;
  if (LMAX >= 1) {
    const float s3 = 1.7320508075688772f;
    Y[1] = s3 * y; Y[2] = s3 * z; Y[3] = s3 * x;
  }
  if (LMAX >= 2) {
    const float s15 = 3.872983346207417f, s5h = 1.118033988749895f;
    Y[4] = s15 * x * y; Y[5] = s15 * y * z; Y[6] = s5h * (3.0f * z * z - 1.0f); Y[7] = s15 * x * z;
    Y[8] = 0.5f * s15 * (x * x - y * y);
  }
  if (LMAX >= 3) {
    const float a = 2.091650066335189f, b = 10.246950765959598f, c = 1.6201851746019651f, s7h = 1.3228756555322954f;
    Y[9] = a * y * (3.0f * x * x - y * y);
    Y[10] = b * x * y * z;
    Y[11] = c * y * (5.0f * z * z - 1.0f);
    Y[12] = s7h * (5.0f * z * z * z - 3.0f * z);
    Y[13] = c * x * (5.0f * z * z - 1.0f);
    Y[14] = 0.5f * b * (x * x - y * y) * z;
    Y[15] = a * x * (x * x - 3.0f * y * y);
  }
}

__device__ __forceinline__ void sph_harm_rt(int lmax, float x, float y, float z, float* Y) {
  switch (lmax) {
    case 0: sph_harm<0>(x, y, z, Y); break;
    case 1: sph_harm<1>(x, y, z, Y); break;
    case 2: sph_harm<2>(x, y, z, Y); break;
    default: sph_harm<3>(x, y, z, Y); break;
  }
}

// t[k] = sum_lm Ybar[lm] * dY_lm/dn_k for the polynomials above (B11; only the tangential part is used).
__device__ __forceinline__ void sph_harm_vjp(int lmax, float x, float y, float z, const float* Yb, float* t) {
  float tx = 0.f, ty = 0.f, tz = 0.f;
  if (lmax >= 1) {
    const float s3 = 1.7320508075688772f;
    ty += s3 * Yb[1]; tz += s3 * Yb[2]; tx += s3 * Yb[3];
  }
  if (lmax >= 2) {
    const float s15 = 3.872983346207417f, s5 = 2.23606797749979f;
    tx += s15 * (y * Yb[4] + z * Yb[7] + x * Yb[8]);
    ty += s15 * (x * Yb[4] + z * Yb[5] - y * Yb[8]);
    tz += s15 * (y * Yb[5] + x * Yb[7]) + 3.0f * s5 * z * Yb[6];
  }
  if (lmax >= 3) {
    const float a = 2.091650066335189f, b = 10.246950765959598f, c = 1.6201851746019651f, s7h = 1.3228756555322954f;
    const float q = 5.0f * z * z - 1.0f;
    tx += a * 6.0f * x * y * Yb[9] + b * y * z * Yb[10] + c * q * Yb[13] + b * x * z * Yb[14] + a * 3.0f * (x * x - y * y) * Yb[15];
    ty += a * 3.0f * (x * x - y * y) * Yb[9] + b * x * z * Yb[10] + c * q * Yb[11] - b * y * z * Yb[14] - a * 6.0f * x * y * Yb[15];
    tz += b * x * y * Yb[10] + c * 10.0f * y * z * Yb[11] + s7h * (15.0f * z * z - 3.0f) * Yb[12] + c * 10.0f * x * z * Yb[13] +
          0.5f * b * (x * x - y * y) * Yb[14];
  }
  t[0] = tx; t[1] = ty; t[2] = tz;
}

// F1 in fp64: u(x) and du/dx for the polynomial envelope of order p, x in [0,1)
__device__ __forceinline__ void envelope_d(double x, int p, double* u, double* dudx) {
  double xp1 = 1.0;  // x^(p-1)
  for (int k = 0; k < p - 1; ++k) xp1 *= x;
  const double xp = xp1 * x;
  const double a = 0.5 * (p + 1) * (p + 2), b = (double)p * (p + 2), c = 0.5 * p * (p + 1);
  *u = 1.0 - a * xp + b * xp * x - c * xp * x * x;
  const double om = 1.0 - x;
  *dudx = -0.5 * p * (p + 1) * (p + 2) * xp1 * om * om;
}

}  // namespace allegro
