// asd_rng.cuh -- in-register thermal noise for the ASD kernels (device only).
//
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11 -- public definition) keyed by (seed; step, global site),
// mapped to three standard normals by Box-Muller.  DESIGN.md readings R1-R3 (PAPER.md P:38 says only
// "normal distribution").  Written independently of oracle/: nothing here is shared with it.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace asd {

// ---- approximate special-function units (MUFU), used where the error budget allows ----
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sin(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_cos(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

struct PhiloxKey {            // the ten round keys are the same for every thread: expanded once on the host
  uint32_t k0[10], k1[10];
};

// One Philox4x32-10 block.  Round: (c0,c1,c2,c3) <- (hi(M1 c2)^c1^k0, lo(M1 c2), hi(M0 c0)^c3^k1, lo(M0 c0)).
__device__ __forceinline__ void philox4x32_10(const PhiloxKey& key, uint32_t c0, uint32_t c1, uint32_t c2,
                                              uint32_t c3, uint32_t r[4]) {
#pragma unroll
  for (int i = 0; i < 10; ++i) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;   // IMAD.WIDE.U32
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ key.k0[i];   // LOP3
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ key.k1[i];
    c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
  }
  r[0] = c0; r[1] = c1; r[2] = c2; r[3] = c3;
}

// R2: u = ((r >> 9) + 1/2) 2^-23 in (0,1), 24 significant bits, formed without an integer->float conversion:
// f = the [1,2) float whose mantissa is r >> 9 (one funnel shift: {0x7F : r} >> 9), u = f - (1 - 2^-24), exact.
__device__ __forceinline__ float unit_float(uint32_t r) { return __uint_as_float(__funnelshift_r(r, 0x7Fu, 9)); }
__device__ __forceinline__ float uniform24(uint32_t r) { return unit_float(r) - 0.99999994039535522461f; }

constexpr float kLnTail = 2.44140625e-4f;   // 2^-12: below this 1 - u, -2 ln u comes from the series

// -2 ln u for u in (0,1) by lg2.approx.  Its absolute error (~2^-22) is harmless except where -2 ln u -> 0, i.e.
// 1 - u < 2^-12; there neg2_ln_tail (the series -ln u = w + w^2/2 + w^3/3, w = 1 - u exact) replaces it.
__device__ __forceinline__ float neg2_ln_fast(float u) { return -1.3862943611198906f * mufu_lg2(u); }
__device__ __forceinline__ float neg2_ln_tail(float w) { return 2.0f * w * fmaf(w, fmaf(w, 0.33333334f, 0.5f), 1.0f); }
__device__ __forceinline__ float neg2_ln(float u) {
  const float w = 1.0f - u;
  return (w < kLnTail) ? neg2_ln_tail(w) : neg2_ln_fast(u);
}

// R3: xi_x = rho0 cos(2 pi u1), xi_y = rho0 sin(2 pi u1), rho0 = sqrt(-2 ln u0); xi_z = rho2 cos(2 pi u3),
// rho2 = sqrt(-2 ln u2).  The angle is shifted to [-pi, pi) for the MUFU range and the sign restored:
// 2 pi (u - 1/2) = 2 pi f - 2 pi (3/2 - 2^-24), one FMA from the [1,2) float.
__device__ __forceinline__ float angle_of(uint32_t r) {
  return fmaf(unit_float(r), 6.283185307179586f, -9.424777586262354f);
}
__device__ __forceinline__ void normals3(const uint32_t r[4], float xi[3]) {
  const float rho0 = mufu_sqrt(neg2_ln(uniform24(r[0])));
  const float rho2 = mufu_sqrt(neg2_ln(uniform24(r[2])));
  const float a1 = angle_of(r[1]), a3 = angle_of(r[3]);
  xi[0] = -rho0 * mufu_cos(a1);
  xi[1] = -rho0 * mufu_sin(a1);
  xi[2] = -rho2 * mufu_cos(a3);
}

// The same for V sites of one thread, with the rare tail of -2 ln u (probability 2^-12 per uniform) moved out of
// the straight-line code: every value first takes the lg2 path, and only a thread that drew a u within 2^-12 of 1
// re-does those values with the series.
template <int V>
__device__ __forceinline__ void normals3_multi(const uint32_t r[V][4], float xi[V][3]) {
  float t0[V], t2[V], wmin = 1.0f;
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float u0 = uniform24(r[v][0]), u2 = uniform24(r[v][2]);
    t0[v] = neg2_ln_fast(u0); t2[v] = neg2_ln_fast(u2);
    wmin = fminf(wmin, 1.0f - fmaxf(u0, u2));
  }
  if (wmin < kLnTail) {
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const float w0 = 1.0f - uniform24(r[v][0]), w2 = 1.0f - uniform24(r[v][2]);
      if (w0 < kLnTail) t0[v] = neg2_ln_tail(w0);
      if (w2 < kLnTail) t2[v] = neg2_ln_tail(w2);
    }
  }
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const float rho0 = mufu_sqrt(t0[v]), rho2 = mufu_sqrt(t2[v]);
    const float a1 = angle_of(r[v][1]), a3 = angle_of(r[v][3]);
    xi[v][0] = -rho0 * mufu_cos(a1);
    xi[v][1] = -rho0 * mufu_sin(a1);
    xi[v][2] = -rho2 * mufu_cos(a3);
  }
}

// R1 counter: (n lo, n hi, g lo, g hi | stream << 28).
__device__ __forceinline__ void philox_site(const PhiloxKey& key, uint32_t n_lo, uint32_t n_hi, uint64_t g,
                                            uint32_t stream, uint32_t r[4]) {
  philox4x32_10(key, n_lo, n_hi, (uint32_t)g, (uint32_t)(g >> 32) | (stream << 28), r);
}

}  // namespace asd
