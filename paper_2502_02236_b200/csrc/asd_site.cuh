// asd_site.cuh -- per-site arithmetic shared by the Heun stage kernels (device only).
//
//   B_i(X) = B_ex + (2 k_u/mu_s)(X_i.e)e + s B_app,i + sigma_i xi_i          Eq. (2),(3)
//   f(S,B) = -gamma/(1+lambda^2) [ S x B + lambda S x (S x B) ]               Eq. (1), in LL form
//   predictor  S~ = normalise(S + dt f),  A = S + dt/2 f
//   corrector  S  = normalise(A + dt/2 f(S~, B(S~)))
#pragma once
#include "asd_rng.cuh"

namespace asd {

struct SiteConst {
  float gdt;      // gamma dt / (1 + lambda^2)
  float lambda;
  float scale;    // B_app = scale * B
};

// q -> q/|q| (0 stays 0: vacant sites and padding hold exact zeros and must keep them).
__device__ __forceinline__ void normalise3(float q0, float q1, float q2, float out[3]) {
  // the floor keeps 1/|q| finite for q = 0 (0 * finite = 0); a real spin has |q| ~ 1
  const float n2 = fmaxf(fmaf(q0, q0, fmaf(q1, q1, q2 * q2)), 1e-30f);
  float inv = mufu_rsqrt(n2);
  inv = inv * fmaf(-0.5f * n2, inv * inv, 1.5f);                  // one Newton step: |S| = 1 to ~1 ulp
  out[0] = q0 * inv; out[1] = q1 * inv; out[2] = q2 * inv;
}

// One site: field assembly, LL torque, update, renormalise.  gp = (e_x, e_y, e_z, 2 k_u/mu_s).
template <int STAGE>
__device__ __forceinline__ void site_update(const SiteConst& p, const float X[3], const float Bex[3],
                                            const float4 gp, const float Bapp[3], float sigma, const float xi[3],
                                            const float Ain[3], float out[3], float outA[3]) {
  const float d = fmaf(X[0], gp.x, fmaf(X[1], gp.y, X[2] * gp.z));
  const float ca = gp.w * d;                                       // Eq. (3): (2 k_u / mu_s)(X.e)
  const float B0 = fmaf(sigma, xi[0], fmaf(p.scale, Bapp[0], fmaf(ca, gp.x, Bex[0])));
  const float B1 = fmaf(sigma, xi[1], fmaf(p.scale, Bapp[1], fmaf(ca, gp.y, Bex[1])));
  const float B2 = fmaf(sigma, xi[2], fmaf(p.scale, Bapp[2], fmaf(ca, gp.z, Bex[2])));
  const float a0 = X[1] * B2 - X[2] * B1, a1 = X[2] * B0 - X[0] * B2, a2 = X[0] * B1 - X[1] * B0;   // S x B
  const float b0 = X[1] * a2 - X[2] * a1, b1 = X[2] * a0 - X[0] * a2, b2 = X[0] * a1 - X[1] * a0;   // S x (S x B)
  const float f0 = -p.gdt * fmaf(p.lambda, b0, a0);               // dt * f(S,B)
  const float f1 = -p.gdt * fmaf(p.lambda, b1, a1);
  const float f2 = -p.gdt * fmaf(p.lambda, b2, a2);
  float q0, q1, q2;
  if (STAGE == 0) {
    outA[0] = fmaf(0.5f, f0, X[0]); outA[1] = fmaf(0.5f, f1, X[1]); outA[2] = fmaf(0.5f, f2, X[2]);
    q0 = X[0] + f0; q1 = X[1] + f1; q2 = X[2] + f2;
  } else {
    q0 = fmaf(0.5f, f0, Ain[0]); q1 = fmaf(0.5f, f1, Ain[1]); q2 = fmaf(0.5f, f2, Ain[2]);
  }
  normalise3(q0, q1, q2, out);
}

}  // namespace asd
