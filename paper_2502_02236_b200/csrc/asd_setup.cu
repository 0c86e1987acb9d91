// asd_setup.cu -- lattice set-up kernels: column table (grain id + in-plane bond mask), per-column anisotropy
// table, dense <-> padded-row conversion of the per-site arrays (asd_internal.cuh), thermal-field amplitude,
// general-ELL transposition.  None of this is on the per-step path.
#include "asd_internal.cuh"

namespace asd {

namespace {

// One thread per track column (gx, j).  A bond to the neighbour column (gx+dx, j+dy) exists iff that column
// exists (periodic wrap in y if pbc_y; in x only if pbc_x, which implies track_nx == nx), is magnetic and has
// the same grain id (exchange-decoupled grains).  flags[0] is raised when two magnetic neighbour columns
// belong to DIFFERENT grains: only then does a kernel need the bond masks (vacant sites hold S = 0 and drop
// out of Eq. (2) by themselves).
// Also writes the per-column copy of the grain's anisotropy (e_x | e_y | e_z | 2 k_u/mu_s), SoA over columns.
__global__ void build_columns_kernel(const int32_t* __restrict__ gmap, uint32_t* __restrict__ col,
                                     const float4* __restrict__ grain, float* __restrict__ aniso,
                                     int32_t* __restrict__ flags, int64_t track_nx, int ny, int pbc_x, int pbc_y) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t ncol = track_nx * ny;
  if (t >= ncol) return;
  const int64_t gx = t / ny;
  const int j = (int)(t - gx * ny);
  const int32_t g = gmap ? gmap[t] : 0;
  const float4 gp = grain[g + 1];                 // entry 0 = vacant
  aniso[t] = gp.x; aniso[ncol + t] = gp.y; aniso[2 * ncol + t] = gp.z; aniso[3 * ncol + t] = gp.w;
  if (g < 0) {                                    // vacant column: id 0; the group flag still has to be right
    uint32_t e0 = 0u;
    const int j4 = j & ~3;
    int32_t first = -1;
    for (int q = j4; q < j4 + 4 && q < ny; ++q) {
      const int32_t gq = gmap[gx * ny + q];
      if (gq < 0) continue;
      if (first < 0) first = gq;
      else if (gq != first) e0 |= COL_GROUP_MIXED;
    }
    col[t] = e0;
    return;
  }
  uint32_t e = (uint32_t)(g + 1) & 0xFFFFu;
  const int dxs[8] = {1, -1, 0, 0, 1, 1, -1, -1};
  const int dys[8] = {0, 0, 1, -1, 1, -1, 1, -1};
  bool touch = false;
#pragma unroll
  for (int b = 0; b < 8; ++b) {
    int64_t x = gx + dxs[b];
    int y = j + dys[b];
    if (x < 0 || x >= track_nx) { if (!pbc_x) continue; x = (x + track_nx) % track_nx; }
    if (y < 0 || y >= ny) { if (!pbc_y) continue; y = (y + ny) % ny; }
    const int32_t gn = gmap ? gmap[x * ny + y] : 0;
    if (gn == g) e |= 1u << (16 + b);
    else if (gn >= 0) touch = true;
  }
  {
    const int j4 = j & ~3;
    int32_t first = -1;
    bool mixed = false;
    for (int q = j4; q < j4 + 4 && q < ny; ++q) {
      const int32_t gq = gmap ? gmap[gx * ny + q] : 0;
      if (gq < 0) continue;
      if (first < 0) first = gq;
      else if (gq != first) mixed = true;
    }
    if (mixed) e |= COL_GROUP_MIXED;
  }
  col[t] = e;
  if (touch) atomicOr(flags, 1);
}

// padded <- dense with vacancy masking (src == nullptr: +z on magnetic sites).  One thread per padded element of
// the real rows: trailing pad elements are (re)written as 0.
__global__ void pack_spins_kernel(const float* __restrict__ sx, const float* __restrict__ sy,
                                  const float* __restrict__ sz, float* __restrict__ dx, float* __restrict__ dy,
                                  float* __restrict__ dz, const uint32_t* __restrict__ col, int64_t nrows, int ny,
                                  int nz, int nyp, int lead) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nrows * nyp) return;
  const int64_t r = t / nyp;
  const int j = (int)(t - r * nyp);
  const int64_t e = t + lead;                      // skip the zero lead
  float vx = 0.0f, vy = 0.0f, vz = 0.0f;
  if (j < ny) {
    const int64_t i = r / nz;
    if ((col[i * ny + j] & 0xFFFFu) != 0u) {
      const int64_t l = r * ny + j;
      vx = sx ? sx[l] : 0.0f; vy = sy ? sy[l] : 0.0f; vz = sz ? sz[l] : 1.0f;
    }
  }
  dx[e] = vx; dy[e] = vy; dz[e] = vz;
}

__global__ void pack_field_kernel(const float* __restrict__ src, float* __restrict__ dst, int64_t nrows, int ny,
                                  int nyp, int lead, float scale, int take_sqrt) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nrows * nyp) return;
  const int64_t r = t / nyp;
  const int j = (int)(t - r * nyp);
  float v = 0.0f;
  if (j < ny) {
    v = src[r * ny + j];
    // sigma_i = c_th sqrt(T_i), c_th = sqrt(2 lambda k_B / (gamma mu_s dt))  [Tesla]  (P:38 with mu_0 absorbed)
    // (T < 0 or NaN gives sigma = 0 instead of a NaN that would spread through the exchange field)
    if (take_sqrt) v = scale * sqrtf(fmaxf(v, 0.0f));
  }
  dst[t + lead] = v;
}

__global__ void unpack_kernel(const float* __restrict__ src, float* __restrict__ dst, int64_t N, int ny, int nyp,
                              int lead) {
  const int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (l >= N) return;
  const int64_t r = l / ny;
  const int j = (int)(l - r * ny);
  dst[l] = src[lead + r * nyp + j];
}

// site-major [N][W] dense site ids -> slot-major [W][N] padded element offsets; J scaled to Tesla.
__global__ void ell_transpose_kernel(const int32_t* __restrict__ idx_in, const float* __restrict__ J_in,
                                     int32_t* __restrict__ idx_out, float* __restrict__ J_out, int64_t N, int W,
                                     int ny, int nyp, int lead, float inv_mu_s_scaled, float j_unit) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= N * W) return;
  const int64_t l = t / W;
  const int s = (int)(t - l * W);
  const int32_t n = idx_in[t];
  // An empty slot is stored as "the site itself with J = 0": the stage kernels then need neither a test nor a select
  // per slot (0 * S_i adds nothing; S_i is finite).
  const bool has = n >= 0 && n < N;
  const int64_t m = has ? (int64_t)n : l;
  const int32_t r = (int32_t)(m / ny);
  idx_out[(int64_t)s * N + l] = lead + r * nyp + (int32_t)(m - (int64_t)r * ny);
  // J/mu_s in Tesla; both factors are far outside fp32 range individually, so rescale first
  J_out[(int64_t)s * N + l] = has ? (J_in[t] * j_unit) * inv_mu_s_scaled : 0.0f;
}

inline unsigned nblocks(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

}  // namespace

asd_status launch_build_columns(Ctx& c) {
  const int64_t n = c.d.track_nx * c.d.ny;
  build_columns_kernel<<<nblocks(n, 256), 256, 0, c.stream>>>(c.grain_map_dev, c.col, c.grain, c.aniso, c.flags,
                                                             c.d.track_nx, c.d.ny, c.d.pbc[0], c.d.pbc[1]);
  ASD_LAUNCH_CHECK(c, "build_columns");
  return ASD_OK;
}

asd_status launch_pack_spins(Ctx& c, CVec3Ptr src, Vec3Ptr dst) {
  const int64_t n = c.nrows * c.nyp;
  pack_spins_kernel<<<nblocks(n, 256), 256, 0, c.stream>>>(src.x, src.y, src.z, dst.x, dst.y, dst.z, c.col_win(),
                                                          c.nrows, c.d.ny, c.d.nz, c.nyp, c.lead);
  ASD_LAUNCH_CHECK(c, "pack_spins");
  return ASD_OK;
}

asd_status launch_pack_field(Ctx& c, const float* dense, float* padded) {
  const int64_t n = c.nrows * c.nyp;
  pack_field_kernel<<<nblocks(n, 256), 256, 0, c.stream>>>(dense, padded, c.nrows, c.d.ny, c.nyp, c.lead, 1.0f, 0);
  ASD_LAUNCH_CHECK(c, "pack_field");
  return ASD_OK;
}

asd_status launch_sigma(Ctx& c, const float* T_dense) {
  const double cth = sqrt(2.0 * c.d.lambda * kBoltzmann / (c.gamma * c.d.mu_s * c.d.dt));
  const int64_t n = c.nrows * c.nyp;
  pack_field_kernel<<<nblocks(n, 256), 256, 0, c.stream>>>(T_dense, c.sigma(), c.nrows, c.d.ny, c.nyp, c.lead, (float)cth, 1);
  ASD_LAUNCH_CHECK(c, "sigma");
  return ASD_OK;
}

asd_status launch_unpack(Ctx& c, const float* padded, float* dense) {
  unpack_kernel<<<nblocks(c.N, 256), 256, 0, c.stream>>>(padded, dense, c.N, c.d.ny, c.nyp, c.lead);
  ASD_LAUNCH_CHECK(c, "unpack");
  return ASD_OK;
}

asd_status launch_ell_transpose(Ctx& c, const int32_t* idx_site_major, const float* J_site_major) {
  const int64_t n = c.N * c.d.ell_width;
  // J ~ 1e-21 J and mu_s ~ 1e-23 J/T: (J * 1e21) * (1e-21 / mu_s) keeps every factor inside fp32 range
  ell_transpose_kernel<<<nblocks(n, 256), 256, 0, c.stream>>>(idx_site_major, J_site_major, c.ell_idx, c.ell_J,
                                                             c.N, c.d.ell_width, c.d.ny, c.nyp, c.lead,
                                                             (float)(1e-21 / c.d.mu_s), 1e21f);
  ASD_LAUNCH_CHECK(c, "ell_transpose");
  return ASD_OK;
}

}  // namespace asd
