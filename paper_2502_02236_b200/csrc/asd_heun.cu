// asd_heun.cu -- the hot path: one fused kernel per stochastic-Heun stage.
//
//   predictor  k1 = f(S, B(S));   S~ = normalise(S + dt k1);   A = S + dt/2 k1
//   corrector  k2 = f(S~, B(S~)); S  = normalise(A + dt/2 k2)          (same xi_i in both stages)
//   f(S,B) = -gamma/(1+lambda^2) [ S x B + lambda S x (S x B) ]        Eq. (1), in LL form
//   B_i(X) = (1/mu_s) sum_j J_ij X_j + (2 k_u/mu_s)(X_i.e)e + s B_app,i + sigma_i xi_i   Eq. (2),(3)
//
// Storing A (12 B/site) instead of k1 lets the corrector run without re-reading S or recomputing k1:
// 52 B (predictor) + 52 B (corrector) = 104 B per site per Heun step.
//
// "direct" variant: each thread owns VEC consecutive sites of one y-row; own row, z+-1 and x+-1 rows are
// read with 128-bit loads, the y+-1 row ends with scalar loads; neighbour reuse is served by L1/L2.
#include "asd_internal.cuh"

namespace asd {

namespace {

constexpr int LAT_SC = 0, LAT_L10 = 1, LAT_ELL = 2;

template <int VEC> struct VecIO;
template <> struct VecIO<1> {
  static __device__ __forceinline__ void ld(const float* p, float v[1]) { v[0] = __ldg(p); }
  static __device__ __forceinline__ void ldu(const uint32_t* p, uint32_t v[1]) { v[0] = __ldg(p); }
  static __device__ __forceinline__ void st(float* p, const float v[1]) { p[0] = v[0]; }
};
template <> struct VecIO<4> {
  static __device__ __forceinline__ void ld(const float* p, float v[4]) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(p));
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
  static __device__ __forceinline__ void ldu(const uint32_t* p, uint32_t v[4]) {
    const uint4 t = __ldg(reinterpret_cast<const uint4*>(p));
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
  static __device__ __forceinline__ void st(float* p, const float v[4]) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
  }
};

// Adds w * (row of one x-plane, y-extended by one site on each side) to the exchange sums.
// ext[c][0] = site j0-1, ext[c][1..VEC] = sites j0..j0+VEC-1, ext[c][VEC+1] = site j0+VEC.
template <int VEC>
struct Row { float e[3][VEC + 2]; };

template <int VEC>
__device__ __forceinline__ void load_row(const StageParams& p, int64_t base, bool row_ok, bool need_l, bool need_r,
                                         int dl, int dr, Row<VEC>& r) {
  // base: index of (row, j0); dl / dr: offsets of the j0-1 / j0+VEC sites relative to base (periodic wrap folded in)
  const float* X[3] = {p.X.x, p.X.y, p.X.z};
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    if (row_ok) VecIO<VEC>::ld(X[c] + base, &r.e[c][1]);
    else {
#pragma unroll
      for (int v = 0; v < VEC; ++v) r.e[c][1 + v] = 0.0f;
    }
    r.e[c][0] = (row_ok && need_l) ? __ldg(X[c] + base + dl) : 0.0f;
    r.e[c][VEC + 1] = (row_ok && need_r) ? __ldg(X[c] + base + dr) : 0.0f;
  }
}

// One site: field assembly, noise, LL torque, update, renormalise.
template <int STAGE>
__device__ __forceinline__ void site_update(const StageParams& p, const float X[3], const float Bex[3],
                                            const float4 gp, const float Bapp[3], float sigma, const float xi[3],
                                            const float Ain[3], float out[3], float outA[3]) {
  const float d = X[0] * gp.x + X[1] * gp.y + X[2] * gp.z;
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
  const float n2 = q0 * q0 + q1 * q1 + q2 * q2;
  float inv = mufu_rsqrt(n2);
  inv = inv * fmaf(-0.5f * n2, inv * inv, 1.5f);                  // one Newton step: |S| = 1 to ~1 ulp
  out[0] = q0 * inv; out[1] = q1 * inv; out[2] = q2 * inv;
}

template <int VEC, int LAT, int STAGE>
__global__ void __launch_bounds__(256) heun_stage_direct(const StageParams p) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t l0 = t * VEC;
  if (l0 >= p.N) return;
  const int l0i = (int)l0;                       // N < 2^31 is enforced at create
  const int i = l0i / p.plane;
  const int pp = l0i - i * p.plane;
  const int k = pp / p.ny;
  const int j0 = pp - k * p.ny;

  uint32_t col[VEC];
  VecIO<VEC>::ldu(p.col + (int64_t)i * p.ny + j0, col);
  bool any = false;
#pragma unroll
  for (int v = 0; v < VEC; ++v) any |= (col[v] & 0xFFFFu) != 0u;
  float o[3][VEC], oA[3][VEC];
  if (!any) {                                    // all vacant: keep the buffers zero there
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int v = 0; v < VEC; ++v) { o[c][v] = 0.0f; oA[c][v] = 0.0f; }
  } else {
    // window edges in x (open boundary): the column table knows only the track ends
    if (!p.pbc_x) {
#pragma unroll
      for (int v = 0; v < VEC; ++v) {
        if (i == p.nx - 1) col[v] &= ~BOND_ALL_XP;
        if (i == 0) col[v] &= ~BOND_ALL_XM;
      }
    }
    float Bex[3][VEC];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int v = 0; v < VEC; ++v) Bex[c][v] = 0.0f;

    Row<VEC> own;
    const int dl = (j0 == 0) ? (p.ny - 1) : -1;                    // j0-1 (wraps only if periodic: else bit clear)
    const int dr = (j0 + VEC == p.ny) ? (VEC - p.ny) : VEC;        // j0+VEC
    if (LAT == LAT_ELL) {
      load_row<VEC>(p, l0, true, false, false, 0, 0, own);
      const float* X[3] = {p.X.x, p.X.y, p.X.z};
      for (int s = 0; s < p.ell_w; ++s) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
          const int64_t e = (int64_t)s * p.N + l0 + v;
          const int32_t n = __ldg(p.ell_idx + e);
          if (n >= 0) {
            const float Jt = __ldg(p.ell_J + e);
#pragma unroll
            for (int c = 0; c < 3; ++c) Bex[c][v] = fmaf(Jt, __ldg(X[c] + n), Bex[c][v]);
          }
        }
      }
    } else {
      const bool needL = (col[0] & (BOND_YM)) != 0u, needR = (col[VEC - 1] & (BOND_YP)) != 0u;
      load_row<VEC>(p, l0, true, needL, needR, dl, dr, own);
      // y +- 1 (shell 1)
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
          const float yp = (col[v] & BOND_YP) ? own.e[c][v + 2] : 0.0f;
          const float ym = (col[v] & BOND_YM) ? own.e[c][v] : 0.0f;
          Bex[c][v] = p.jx[0] * (yp + ym);
        }
      // z +- 1 (SC: shell 1; L1_0: shell 2) -- same column, so always the same grain
      {
        const float jz = (LAT == LAT_SC) ? p.jx[0] : p.jx[1];
        const bool zp_ok = (k < p.nz - 1) || p.pbc_z, zm_ok = (k > 0) || p.pbc_z;
        const int dzp = (k == p.nz - 1) ? -(p.nz - 1) * p.ny : p.ny;
        const int dzm = (k == 0) ? (p.nz - 1) * p.ny : -p.ny;
        Row<VEC> zr;
        load_row<VEC>(p, l0 + dzp, zp_ok, false, false, 0, 0, zr);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
          for (int v = 0; v < VEC; ++v) Bex[c][v] = fmaf(jz, zr.e[c][v + 1], Bex[c][v]);
        load_row<VEC>(p, l0 + dzm, zm_ok, false, false, 0, 0, zr);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
          for (int v = 0; v < VEC; ++v) Bex[c][v] = fmaf(jz, zr.e[c][v + 1], Bex[c][v]);
      }
      // x +- 1 (shell 1) and, for L1_0, the in-plane diagonals (shell 3)
#pragma unroll
      for (int side = 0; side < 2; ++side) {
        const uint32_t bX = side == 0 ? BOND_XP : BOND_XM;
        const uint32_t bXYP = side == 0 ? BOND_XPYP : BOND_XMYP;
        const uint32_t bXYM = side == 0 ? BOND_XPYM : BOND_XMYM;
        const int64_t dx = side == 0 ? ((i == p.nx - 1) ? -(int64_t)(p.nx - 1) * p.plane : (int64_t)p.plane)
                                     : ((i == 0) ? (int64_t)(p.nx - 1) * p.plane : -(int64_t)p.plane);
        uint32_t anyb = 0u;
#pragma unroll
        for (int v = 0; v < VEC; ++v) anyb |= col[v];
        const bool row_ok = (anyb & (bX | bXYP | bXYM)) != 0u;
        const bool nl = (LAT == LAT_L10) && (col[0] & bXYM) != 0u;
        const bool nr = (LAT == LAT_L10) && (col[VEC - 1] & bXYP) != 0u;
        Row<VEC> xr;
        load_row<VEC>(p, l0 + dx, row_ok, nl, nr, dl, dr, xr);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
          for (int v = 0; v < VEC; ++v) {
            const float xs = (col[v] & bX) ? xr.e[c][v + 1] : 0.0f;
            Bex[c][v] = fmaf(p.jx[0], xs, Bex[c][v]);
            if (LAT == LAT_L10) {
              const float dp = (col[v] & bXYP) ? xr.e[c][v + 2] : 0.0f;
              const float dm = (col[v] & bXYM) ? xr.e[c][v] : 0.0f;
              Bex[c][v] = fmaf(p.jx[2], dp + dm, Bex[c][v]);
            }
          }
      }
    }

    float sg[VEC], Ba[3][VEC], Ain[3][VEC];
    VecIO<VEC>::ld(p.sigma + l0, sg);
    VecIO<VEC>::ld(p.Bx + l0, Ba[0]);
    VecIO<VEC>::ld(p.By + l0, Ba[1]);
    VecIO<VEC>::ld(p.Bz + l0, Ba[2]);
    if (STAGE == 1) {
      VecIO<VEC>::ld(p.A.x + l0, Ain[0]);
      VecIO<VEC>::ld(p.A.y + l0, Ain[1]);
      VecIO<VEC>::ld(p.A.z + l0, Ain[2]);
    }
    const uint64_t g = p.g0 + (uint64_t)l0;
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
      const uint32_t gid = col[v] & 0xFFFFu;
      if (gid == 0u) {
        o[0][v] = o[1][v] = o[2][v] = 0.0f;
        oA[0][v] = oA[1][v] = oA[2][v] = 0.0f;
        continue;
      }
      uint32_t r[4];
      philox_site(p.key, p.n_lo, p.n_hi, g + v, 0u, r);
      float xi[3];
      normals3(r, xi);
      const float4 gp = __ldg(p.grain + (gid - 1u));
      const float X[3] = {own.e[0][v + 1], own.e[1][v + 1], own.e[2][v + 1]};
      const float Be[3] = {Bex[0][v], Bex[1][v], Bex[2][v]};
      const float Bap[3] = {Ba[0][v], Ba[1][v], Ba[2][v]};
      const float Ai[3] = {Ain[0][v], Ain[1][v], Ain[2][v]};
      float ov[3], oAv[3];
      site_update<STAGE>(p, X, Be, gp, Bap, sg[v], xi, Ai, ov, oAv);
      o[0][v] = ov[0]; o[1][v] = ov[1]; o[2][v] = ov[2];
      if (STAGE == 0) { oA[0][v] = oAv[0]; oA[1][v] = oAv[1]; oA[2][v] = oAv[2]; }
    }
  }
  VecIO<VEC>::st(p.out.x + l0, o[0]);
  VecIO<VEC>::st(p.out.y + l0, o[1]);
  VecIO<VEC>::st(p.out.z + l0, o[2]);
  if (STAGE == 0) {
    VecIO<VEC>::st(p.outA.x + l0, oA[0]);
    VecIO<VEC>::st(p.outA.y + l0, oA[1]);
    VecIO<VEC>::st(p.outA.z + l0, oA[2]);
  }
}

template <int VEC, int LAT>
asd_status launch_pair(Ctx& c, StageParams& p) {
  const int threads = 256;
  const int64_t nthreads = (c.N + VEC - 1) / VEC;
  const unsigned blocks = (unsigned)((nthreads + threads - 1) / threads);
  // predictor: X = S -> out = S~, outA = A
  p.X = {c.S.x, c.S.y, c.S.z};
  p.out = c.St; p.outA = c.A; p.A = {nullptr, nullptr, nullptr};
  heun_stage_direct<VEC, LAT, 0><<<blocks, threads, 0, c.stream>>>(p);
  ASD_LAUNCH_CHECK(c, "heun predictor");
  // corrector: X = S~, A -> out = S
  p.X = {c.St.x, c.St.y, c.St.z};
  p.A = {c.A.x, c.A.y, c.A.z};
  p.out = c.S; p.outA = {nullptr, nullptr, nullptr};
  heun_stage_direct<VEC, LAT, 1><<<blocks, threads, 0, c.stream>>>(p);
  ASD_LAUNCH_CHECK(c, "heun corrector");
  return ASD_OK;
}

}  // namespace

void fill_stage_params(const Ctx& c, StageParams& p) {
  p.sigma = c.sigma; p.Bx = c.Bx; p.By = c.By; p.Bz = c.Bz;
  p.col = c.col + c.x0 * c.d.ny;
  p.grain = c.grain;
  p.ell_idx = c.ell_idx; p.ell_J = c.ell_J; p.ell_w = c.d.ell_width;
  p.nx = c.d.nx; p.ny = c.d.ny; p.nz = c.d.nz; p.plane = c.plane; p.N = c.N;
  p.pbc_x = c.d.pbc[0]; p.pbc_y = c.d.pbc[1]; p.pbc_z = c.d.pbc[2];
  for (int a = 0; a < 3; ++a) p.jx[a] = (float)(c.d.J[a] / c.d.mu_s);
  p.gdt = (float)(c.gamma * c.d.dt / (1.0 + c.d.lambda * c.d.lambda));
  p.lambda = (float)c.d.lambda;
  p.scale = c.scale;
  p.g0 = (uint64_t)c.x0 * (uint64_t)c.plane;
  uint32_t k0 = (uint32_t)(c.d.seed & 0xFFFFFFFFull), k1 = (uint32_t)(c.d.seed >> 32);
  for (int r = 0; r < 10; ++r) {
    p.key.k0[r] = k0; p.key.k1[r] = k1;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
}

asd_status launch_heun(Ctx& c, int64_t n) {
  StageParams p;
  fill_stage_params(c, p);
  const bool vec4 = (c.d.ny % 4 == 0);
  for (int64_t s = 0; s < n; ++s) {
    p.n_lo = (uint32_t)((uint64_t)c.step & 0xFFFFFFFFull);
    p.n_hi = (uint32_t)((uint64_t)c.step >> 32);
    asd_status st;
    if (c.d.ell_width > 0) st = launch_pair<1, LAT_ELL>(c, p);
    else if (c.d.lattice == ASD_SC) st = vec4 ? launch_pair<4, LAT_SC>(c, p) : launch_pair<1, LAT_SC>(c, p);
    else st = vec4 ? launch_pair<4, LAT_L10>(c, p) : launch_pair<1, LAT_L10>(c, p);
    if (st != ASD_OK) return st;
    c.step += 1;
  }
  return ASD_OK;
}

}  // namespace asd
