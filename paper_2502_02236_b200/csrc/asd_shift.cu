// asd_shift.cu -- the moving-window shift.
//
//   1. outgoing planes i < p : out_sum[c] += S_i, out_cnt[c] += 1 over magnetic sites (Eq. (6) with mu_S/V
//      factored out), one warp per macrocell, lanes in ascending site order, warp-shuffle reduction in fp64
//   2. move                  : S(i,.,.) <- S(i+p,.,.) -- written into the scratch buffer S~, then S and S~ swap
//   3. incoming planes       : vacant columns 0; magnetic sites drawn in a cone about the track magnetisation of
//      their macrocell, polar angle uniform on [0, theta_max], sin(theta_max)/theta_max = M/M_S^0 (D:S3)
//   4. x0 += p (the column table is track-wide, so nothing else follows the window)
#include "asd_internal.cuh"

namespace asd {

namespace {

struct ShiftGeom {
  int nx, ny, nz, plane;   // plane = ny*nz (dense)
  int nyp, lead;           // padded-row layout (asd_internal.cuh)
  int mx, my, mz;
  int64_t x0;           // window origin BEFORE the shift
  int64_t ncy, ncz;
  int p;
};

// One warp per macrocell touching the outgoing slab [x0, x0+p).
__global__ void coarse_grain_outgoing(const float* __restrict__ sx, const float* __restrict__ sy,
                                      const float* __restrict__ sz, const uint32_t* __restrict__ col_track,
                                      double* __restrict__ out_sum, long long* __restrict__ out_cnt, ShiftGeom g,
                                      int64_t cx_first, int n_cx) {
  const int warp = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  const int64_t ncell_slab = (int64_t)n_cx * g.ncy * g.ncz;
  if (warp >= ncell_slab) return;                       // whole warps exit together
  const int cz = (int)(warp % g.ncz);
  const int cy = (int)((warp / g.ncz) % g.ncy);
  const int64_t cx = cx_first + warp / (g.ncz * g.ncy);
  // cell extent intersected with the slab and the lattice
  const int64_t gx_lo = max(cx * g.mx, g.x0), gx_hi = min((cx + 1) * (int64_t)g.mx, g.x0 + g.p);
  const int j_lo = cy * g.my, j_hi = min((cy + 1) * g.my, g.ny);
  const int k_lo = cz * g.mz, k_hi = min((cz + 1) * g.mz, g.nz);
  const int ni = (int)(gx_hi - gx_lo), nj = j_hi - j_lo, nk = k_hi - k_lo;
  const int total = ni * nk * nj;
  double s0 = 0.0, s1 = 0.0, s2 = 0.0;
  long long cnt = 0;
  for (int q = lane; q < total; q += 32) {              // q ascends with l = (i*nz + k)*ny + j
    const int dj = q % nj, dk = (q / nj) % nk, di = q / (nj * nk);
    const int64_t gx = gx_lo + di;
    const int j = j_lo + dj, k = k_lo + dk;
    if ((col_track[gx * g.ny + j] & 0xFFFFu) == 0u) continue;
    const int64_t l = g.lead + ((gx - g.x0) * g.nz + k) * (int64_t)g.nyp + j;
    s0 += (double)sx[l]; s1 += (double)sy[l]; s2 += (double)sz[l];
    cnt += 1;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    s0 += __shfl_down_sync(0xffffffffu, s0, off);
    s1 += __shfl_down_sync(0xffffffffu, s1, off);
    s2 += __shfl_down_sync(0xffffffffu, s2, off);
    cnt += __shfl_down_sync(0xffffffffu, cnt, off);
  }
  if (lane == 0) {
    const int64_t c = (cx * g.ncy + cy) * g.ncz + cz;
    out_sum[3 * c] += s0; out_sum[3 * c + 1] += s1; out_sum[3 * c + 2] += s2;
    out_cnt[c] += cnt;
  }
}

// dst[l] = src[l + off] for l < n_keep, three components.
__global__ void move_planes_v4(const float4* __restrict__ sx, const float4* __restrict__ sy,
                               const float4* __restrict__ sz, float4* __restrict__ dx, float4* __restrict__ dy,
                               float4* __restrict__ dz, int64_t off4, int64_t n_keep4) {
  const int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (l >= n_keep4) return;
  dx[l] = sx[l + off4]; dy[l] = sy[l + off4]; dz[l] = sz[l + off4];
}

// One thread per site of the incoming planes (window planes nx-p .. nx-1 AFTER the move).
__global__ void seed_incoming(float* __restrict__ dx, float* __restrict__ dy, float* __restrict__ dz,
                              const uint32_t* __restrict__ col_track, const float* __restrict__ cell_frame,
                              ShiftGeom g, PhiloxKey key, uint32_t pass_lo, uint32_t pass_hi, int64_t cx_sub = 0) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (int64_t)g.p * g.plane) return;
  const int di = (int)(t / g.plane);
  const int pp = (int)(t - (int64_t)di * g.plane);
  const int k = pp / g.ny, j = pp - k * g.ny;
  const int i = g.nx - g.p + di;                       // window plane after the move
  const int64_t gx = g.x0 + g.p + i;                   // its global plane
  const int64_t l = g.lead + ((int64_t)i * g.nz + k) * g.nyp + j;
  if ((col_track[gx * g.ny + j] & 0xFFFFu) == 0u) { dx[l] = 0.0f; dy[l] = 0.0f; dz[l] = 0.0f; return; }
  // cell_frame is indexed by track macrocell, or (cx_sub != 0) by the cells of the mesh columns the planes come from
  const int64_t c = ((gx / g.mx - cx_sub) * g.ncy + (j / g.my)) * g.ncz + (k / g.mz);
  const float* f = cell_frame + 12 * c;
  const float theta_max = f[0];
  uint32_t r[4];
  const uint64_t gid = (uint64_t)((gx * g.nz + k) * g.ny + j);
  philox_site(key, pass_lo, pass_hi, gid, 1u, r);
  const float theta = theta_max * uniform24(r[0]);
  const float phi = 6.283185307179586f * uniform24(r[1]);
  float st, ct, sp, cp;
  sincosf(theta, &st, &ct);
  sincosf(phi, &sp, &cp);
  const float a = st * cp, b = st * sp;
  dx[l] = a * f[4] + b * f[7] + ct * f[1];
  dy[l] = a * f[5] + b * f[8] + ct * f[2];
  dz[l] = a * f[6] + b * f[9] + ct * f[3];
}

// One thread per track macrocell: theta_max and the orthonormal frame (n, e1, e2) of its initial magnetisation.
__global__ void cell_frames_kernel(const float* __restrict__ init_mean, float* __restrict__ cell_frame,
                                   int64_t ncell) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  const double v0 = init_mean[3 * c], v1 = init_mean[3 * c + 1], v2 = init_mean[3 * c + 2];
  const double vn = sqrt(v0 * v0 + v1 * v1 + v2 * v2);
  const double m = fmin(1.0, vn);
  double n0 = 0.0, n1 = 0.0, n2 = 1.0;
  if (vn > 0.0) { n0 = v0 / vn; n1 = v1 / vn; n2 = v2 / vn; }
  // e1 = normalise(n x x^) = (0, n_z, -n_y), or n x y^ = (-n_z, 0, n_x) when n is close to x^
  double a0, a1, a2;
  if (fabs(n0) > 0.9) { a0 = -n2; a1 = 0.0; a2 = n0; } else { a0 = 0.0; a1 = n2; a2 = -n1; }
  const double an = sqrt(a0 * a0 + a1 * a1 + a2 * a2);
  a0 /= an; a1 /= an; a2 /= an;
  const double b0 = n1 * a2 - n2 * a1, b1 = n2 * a0 - n0 * a2, b2 = n0 * a1 - n1 * a0;   // e2 = n x e1
  // theta_max: root in [0, pi] of sin(t)/t = m (monotone decreasing), by bisection
  double th;
  if (m >= 1.0) th = 0.0;
  else if (m <= 0.0) th = 3.14159265358979323846;
  else {
    double lo = 0.0, hi = 3.14159265358979323846;
    for (int it = 0; it < 60; ++it) {
      const double mid = 0.5 * (lo + hi);
      if (sin(mid) > m * mid) lo = mid; else hi = mid;
    }
    th = 0.5 * (lo + hi);
  }
  float* f = cell_frame + 12 * c;
  f[0] = (float)th;
  f[1] = (float)n0; f[2] = (float)n1; f[3] = (float)n2;
  f[4] = (float)a0; f[5] = (float)a1; f[6] = (float)a2;
  f[7] = (float)b0; f[8] = (float)b1; f[9] = (float)b2;
  f[10] = 0.0f; f[11] = 0.0f;
}

// End of a pass (reading T1): what the pass has written becomes what lies ahead of the next one.
__global__ void track_commit_kernel(const double* __restrict__ out_sum, const long long* __restrict__ out_cnt,
                                    float* __restrict__ init_mean, int64_t ncell) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  const long long n = out_cnt[c];
  if (n == 0) return;                                   // never written: keeps its value
  const double inv = 1.0 / (double)n;
  init_mean[3 * c] = (float)(out_sum[3 * c] * inv);
  init_mean[3 * c + 1] = (float)(out_sum[3 * c + 1] * inv);
  init_mean[3 * c + 2] = (float)(out_sum[3 * c + 2] * inv);
}

// Read-back scan (reading T3): one CTA per reader position; thread t takes the (cx, cy) cell columns t, t + 256, ...
// in ascending order and the partial sums meet in a fixed tree, so the result does not depend on scheduling.
constexpr int kScanThreads = 256;
__global__ void __launch_bounds__(kScanThreads)
track_read_scan_kernel(const double* __restrict__ out_sum, const long long* __restrict__ out_cnt, int64_t ncx,
                       int64_t ncy, int64_t ncz, int mx, int my, double y_r, double inv2sx, double inv2sy,
                       double x_first, double x_step, double* __restrict__ out) {
  __shared__ double s_num[kScanThreads], s_den[kScanThreads];
  const double x_r = x_first + (double)blockIdx.x * x_step;
  double num = 0.0, den = 0.0;
  for (int64_t q = threadIdx.x; q < ncx * ncy; q += kScanThreads) {
    const int64_t cx = q / ncy, cy = q - cx * ncy;
    const double dx = ((double)cx + 0.5) * mx - x_r, dy = ((double)cy + 0.5) * my - y_r;
    const double w = exp(-dx * dx * inv2sx - dy * dy * inv2sy);
    if (w == 0.0) continue;
    for (int64_t cz = 0; cz < ncz; ++cz) {
      const int64_t c = q * ncz + cz;
      num += w * out_sum[3 * c + 2];
      den += w * (double)out_cnt[c];
    }
  }
  s_num[threadIdx.x] = num; s_den[threadIdx.x] = den;
  __syncthreads();
  for (int off = kScanThreads / 2; off > 0; off >>= 1) {
    if ((int)threadIdx.x < off) { s_num[threadIdx.x] += s_num[threadIdx.x + off]; s_den[threadIdx.x] += s_den[threadIdx.x + off]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) out[blockIdx.x] = s_den[0] > 0.0 ? s_num[0] / s_den[0] : 0.0;
}

inline unsigned nblocks(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

ShiftGeom shift_geom(const Ctx& c, int p) {
  ShiftGeom g;
  g.nx = c.d.nx; g.ny = c.d.ny; g.nz = c.d.nz; g.plane = c.plane; g.nyp = c.nyp; g.lead = c.lead;
  g.mx = c.d.macro[0]; g.my = c.d.macro[1]; g.mz = c.d.macro[2];
  g.x0 = c.x0; g.ncy = c.ncy; g.ncz = c.ncz; g.p = p;
  return g;
}

PhiloxKey expand_key(uint64_t seed) {
  PhiloxKey key;
  uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { key.k0[r] = k0; key.k1[r] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
  return key;
}

// Eq. (6) over window planes [0, p): the macrocells they touch accumulate the spins and the site counts.
asd_status launch_coarse_grain(Ctx& c, const ShiftGeom& g) {
  const Vec3Ptr S = c.S();
  const int64_t cx_first = c.x0 / g.mx, cx_last = (c.x0 + g.p - 1) / g.mx;
  const int n_cx = (int)(cx_last - cx_first + 1);
  const int64_t warps = (int64_t)n_cx * c.ncy * c.ncz;
  coarse_grain_outgoing<<<nblocks(warps * 32, 256), 256, 0, c.stream>>>(S.x, S.y, S.z, c.col, c.out_sum,
                                                                       c.out_cnt, g, cx_first, n_cx);
  ASD_LAUNCH_CHECK(c, "coarse_grain_outgoing");
  return ASD_OK;
}

}  // namespace

// asd_track_end_pass: all nx planes of the window -> track (Eq. (6)); written cells -> init_mean; frames rebuilt.
asd_status launch_track_end_pass(Ctx& c) {
  if (c.mm) { const asd_status sm = mm_flush_to_track(c); if (sm != ASD_OK) return sm; }
  const asd_status st = launch_coarse_grain(c, shift_geom(c, c.d.nx));
  if (st != ASD_OK) return st;
  track_commit_kernel<<<nblocks(c.ncell, 128), 128, 0, c.stream>>>(c.out_sum, c.out_cnt, c.init_mean, c.ncell);
  ASD_LAUNCH_CHECK(c, "track_commit");
  return launch_cell_frames(c);
}

// asd_track_begin_pass: written store cleared; pass += 1; window at x0_new; every plane seeded from the track.
asd_status launch_track_begin_pass(Ctx& c, int64_t x0_new) {
  ASD_CUDA_TRY(c, cudaMemsetAsync(c.out_sum, 0, sizeof(double) * 3 * (size_t)c.ncell, c.stream));
  ASD_CUDA_TRY(c, cudaMemsetAsync(c.out_cnt, 0, sizeof(long long) * (size_t)c.ncell, c.stream));
  c.pass += 1;
  c.x0 = x0_new;
  ShiftGeom g = shift_geom(c, c.d.nx);
  g.x0 = x0_new - c.d.nx;                               // seed_incoming's planes nx-p .. nx-1 "after a shift by p" = all of them
  const Vec3Ptr S = c.S();
  seed_incoming<<<nblocks((int64_t)c.d.nx * c.plane, 256), 256, 0, c.stream>>>(
      S.x, S.y, S.z, c.col, c.cell_frame, g, expand_key(c.d.seed), (uint32_t)((uint64_t)c.pass & 0xFFFFFFFFull),
      (uint32_t)((uint64_t)c.pass >> 32));
  ASD_LAUNCH_CHECK(c, "seed_incoming(all planes)");
  if (c.mm) return mm_restart_from_track(c);
  return ASD_OK;
}

// asd_track_read_scan: `count` reader positions into HOST out; synchronises.  The device results land in the
// reduction scratch (4 * kMaxPartialBlocks doubles), so long scans go in chunks.
asd_status launch_track_read_scan(Ctx& c, double y_r, double sigma_x, double sigma_y, double x_first, double x_step,
                                  int64_t count, double* out_host) {
  const int64_t chunk = 4 * (int64_t)kMaxPartialBlocks;
  for (int64_t done = 0; done < count; done += chunk) {
    const int64_t n = count - done < chunk ? count - done : chunk;
    track_read_scan_kernel<<<(unsigned)n, kScanThreads, 0, c.stream>>>(
        c.out_sum, c.out_cnt, c.ncx, c.ncy, c.ncz, c.d.macro[0], c.d.macro[1], y_r, 0.5 / (sigma_x * sigma_x),
        0.5 / (sigma_y * sigma_y), x_first + (double)done * x_step, x_step, c.partials);
    ASD_LAUNCH_CHECK(c, "track_read_scan");
    ASD_CUDA_TRY(c, cudaMemcpyAsync(out_host + done, c.partials, sizeof(double) * (size_t)n, cudaMemcpyDeviceToHost, c.stream));
    ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  }
  return ASD_OK;
}

asd_status launch_cell_frames(Ctx& c) {
  cell_frames_kernel<<<nblocks(c.ncell, 128), 128, 0, c.stream>>>(c.init_mean, c.cell_frame, c.ncell);
  ASD_LAUNCH_CHECK(c, "cell_frames");
  return ASD_OK;
}

// Shift of a multiscale window by p = pc * mx planes (reading M10; Fig. 1 of the paper): trailing mesh
// -> track, outgoing atoms -> trailing mesh (Eq. (6)), atoms move, leading mesh -> incoming atoms (cone about m with
// magnitude m_e), both meshes move, track ahead -> leading mesh.
asd_status launch_shift_mm(Ctx& c, int32_t p) {
  const int pc = p / c.d.macro[0];
  { const asd_status st = mm_shift_prepare(c, pc); if (st != ASD_OK) return st; }
  const ShiftGeom g = shift_geom(c, p);
  const Vec3Ptr S = c.S(), St = c.St();
  const int64_t planep = (int64_t)c.d.nz * c.nyp;
  const int64_t off = (int64_t)p * planep, n_keep = c.nrows * c.nyp - off;
  if (n_keep > 0) {
    move_planes_v4<<<nblocks(n_keep / 4, 256), 256, 0, c.stream>>>(
        (const float4*)(S.x + c.lead), (const float4*)(S.y + c.lead), (const float4*)(S.z + c.lead),
        (float4*)(St.x + c.lead), (float4*)(St.y + c.lead), (float4*)(St.z + c.lead), off / 4, n_keep / 4);
    ASD_LAUNCH_CHECK(c, "move_planes");
  }
  seed_incoming<<<nblocks((int64_t)p * c.plane, 256), 256, 0, c.stream>>>(
      St.x, St.y, St.z, c.col, mm_shift_frames(c), g, expand_key(c.d.seed), (uint32_t)((uint64_t)c.pass & 0xFFFFFFFFull),
      (uint32_t)((uint64_t)c.pass >> 32), (c.x0 + c.d.nx) / c.d.macro[0]);
  ASD_LAUNCH_CHECK(c, "seed_incoming(from the leading mesh)");
  { const asd_status st = mm_shift_finish(c, pc); if (st != ASD_OK) return st; }   // still at the old window origin
  { const int t = c.aS; c.aS = c.aSt; c.aSt = t; }
  c.x0 += p;
  c.shift += 1;
  return ASD_OK;
}

asd_status launch_shift(Ctx& c, int32_t p) {
  const ShiftGeom g = shift_geom(c, p);
  const Vec3Ptr S = c.S(), St = c.St();
  // 1. outgoing slab -> macrocells
  { const asd_status st = launch_coarse_grain(c, g); if (st != ASD_OK) return st; }
  // 2. move into the scratch buffer
  // (padded planes: nz*nyp floats each, a multiple of 4; the pads move with their rows and stay zero)
  const int64_t planep = (int64_t)c.d.nz * c.nyp;
  const int64_t off = (int64_t)p * planep, n_keep = c.nrows * c.nyp - off;
  if (n_keep > 0) {
    move_planes_v4<<<nblocks(n_keep / 4, 256), 256, 0, c.stream>>>(
        (const float4*)(S.x + c.lead), (const float4*)(S.y + c.lead), (const float4*)(S.z + c.lead),
        (float4*)(St.x + c.lead), (float4*)(St.y + c.lead), (float4*)(St.z + c.lead), off / 4, n_keep / 4);
    ASD_LAUNCH_CHECK(c, "move_planes");
  }
  // 3. incoming slab
  const PhiloxKey key = expand_key(c.d.seed);
  seed_incoming<<<nblocks((int64_t)p * c.plane, 256), 256, 0, c.stream>>>(
      St.x, St.y, St.z, c.col, c.cell_frame, g, key, (uint32_t)((uint64_t)c.pass & 0xFFFFFFFFull),
      (uint32_t)((uint64_t)c.pass >> 32));
  ASD_LAUNCH_CHECK(c, "seed_incoming");
  // 4. swap and advance
  { const int t = c.aS; c.aS = c.aSt; c.aSt = t; }
  c.x0 += p;
  c.shift += 1;
  return ASD_OK;
}

}  // namespace asd
