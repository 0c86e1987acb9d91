// asd_setup.cu -- lattice set-up kernels: column table (grain id + in-plane bond mask), spin masking,
// thermal-field amplitude, general-ELL transposition.  None of this is on the per-step path.
#include "asd_internal.cuh"

namespace asd {

namespace {

// One thread per track column (gx, j).  A bond to the neighbour column (gx+dx, j+dy) exists iff that column
// exists (periodic wrap in y if pbc_y; in x only if pbc_x, which implies track_nx == nx), is magnetic and has
// the same grain id (exchange-decoupled grains).
__global__ void build_columns_kernel(const int32_t* __restrict__ gmap, uint32_t* __restrict__ col, int64_t track_nx,
                                     int ny, int pbc_x, int pbc_y) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= track_nx * ny) return;
  const int64_t gx = t / ny;
  const int j = (int)(t - gx * ny);
  const int32_t g = gmap ? gmap[t] : 0;
  if (g < 0) { col[t] = 0u; return; }
  uint32_t e = (uint32_t)(g + 1) & 0xFFFFu;
  const int dxs[8] = {1, -1, 0, 0, 1, 1, -1, -1};
  const int dys[8] = {0, 0, 1, -1, 1, -1, 1, -1};
#pragma unroll
  for (int b = 0; b < 8; ++b) {
    int64_t x = gx + dxs[b];
    int y = j + dys[b];
    if (x < 0 || x >= track_nx) { if (!pbc_x) continue; x = (x + track_nx) % track_nx; }
    if (y < 0 || y >= ny) { if (!pbc_y) continue; y = (y + ny) % ny; }
    const int32_t gn = gmap ? gmap[x * ny + y] : 0;
    if (gn == g) e |= 1u << (16 + b);
  }
  col[t] = e;
}

// dst = src on magnetic sites, 0 on vacant ones (src == nullptr: +z on magnetic sites).
__global__ void mask_spins_kernel(const float* __restrict__ sx, const float* __restrict__ sy,
                                  const float* __restrict__ sz, float* __restrict__ dx, float* __restrict__ dy,
                                  float* __restrict__ dz, const uint32_t* __restrict__ col, int64_t N, int plane,
                                  int ny) {
  const int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (l >= N) return;
  const int64_t i = l / plane;
  const int j = (int)((l - i * plane) % ny);
  const bool mag = (col[i * ny + j] & 0xFFFFu) != 0u;
  dx[l] = mag ? (sx ? sx[l] : 0.0f) : 0.0f;
  dy[l] = mag ? (sy ? sy[l] : 0.0f) : 0.0f;
  dz[l] = mag ? (sz ? sz[l] : 1.0f) : 0.0f;
}

// sigma_i = c_th sqrt(T_i), c_th = sqrt(2 lambda k_B / (gamma mu_s dt))  [Tesla]  (P:38 with mu_0 absorbed)
__global__ void sigma_kernel(const float* __restrict__ T, float* __restrict__ sigma, int64_t N, float c_th) {
  const int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (l < N) sigma[l] = c_th * sqrtf(T[l]);
}

// site-major [N][W] -> slot-major [W][N]; J scaled to Tesla.
__global__ void ell_transpose_kernel(const int32_t* __restrict__ idx_in, const float* __restrict__ J_in,
                                     int32_t* __restrict__ idx_out, float* __restrict__ J_out, int64_t N, int W,
                                     float inv_mu_s_scaled, float j_unit) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= N * W) return;
  const int64_t l = t / W;
  const int s = (int)(t - l * W);
  const int32_t n = idx_in[t];
  idx_out[(int64_t)s * N + l] = (n >= 0 && n < N) ? n : -1;
  // J/mu_s in Tesla; both factors are far outside fp32 range individually, so rescale first
  J_out[(int64_t)s * N + l] = (J_in[t] * j_unit) * inv_mu_s_scaled;
}

inline unsigned nblocks(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

}  // namespace

asd_status launch_build_columns(Ctx& c) {
  const int64_t n = c.d.track_nx * c.d.ny;
  build_columns_kernel<<<nblocks(n, 256), 256, 0, c.stream>>>(c.grain_map_dev, c.col, c.d.track_nx, c.d.ny,
                                                             c.d.pbc[0], c.d.pbc[1]);
  ASD_LAUNCH_CHECK(c, "build_columns");
  return ASD_OK;
}

asd_status launch_mask_spins(Ctx& c, CVec3Ptr src, Vec3Ptr dst) {
  mask_spins_kernel<<<nblocks(c.N, 256), 256, 0, c.stream>>>(src.x, src.y, src.z, dst.x, dst.y, dst.z,
                                                            c.col + c.x0 * c.d.ny, c.N, c.plane, c.d.ny);
  ASD_LAUNCH_CHECK(c, "mask_spins");
  return ASD_OK;
}

asd_status launch_init_spins(Ctx& c) {
  return launch_mask_spins(c, CVec3Ptr{nullptr, nullptr, nullptr}, c.S);
}

asd_status launch_sigma(Ctx& c, const float* T_dev) {
  const double cth = sqrt(2.0 * c.d.lambda * kBoltzmann / (c.gamma * c.d.mu_s * c.d.dt));
  sigma_kernel<<<nblocks(c.N, 256), 256, 0, c.stream>>>(T_dev, c.sigma, c.N, (float)cth);
  ASD_LAUNCH_CHECK(c, "sigma");
  return ASD_OK;
}

asd_status launch_ell_transpose(Ctx& c, const int32_t* idx_site_major, const float* J_site_major) {
  const int64_t n = c.N * c.d.ell_width;
  // J ~ 1e-21 J and mu_s ~ 1e-23 J/T: (J * 1e21) * (1e-21 / mu_s) keeps every factor inside fp32 range
  ell_transpose_kernel<<<nblocks(n, 256), 256, 0, c.stream>>>(idx_site_major, J_site_major, c.ell_idx, c.ell_J,
                                                             c.N, c.d.ell_width, (float)(1e-21 / c.d.mu_s), 1e21f);
  ASD_LAUNCH_CHECK(c, "ell_transpose");
  return ASD_OK;
}

}  // namespace asd
