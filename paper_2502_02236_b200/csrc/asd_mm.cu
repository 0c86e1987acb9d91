// asd_mm.cu -- the multiscale window (Fig. 1):
// a micromagnetic LLG mesh either side of the atomistic mesh, exchange coupled to it across the mesh boundaries, all
// three moving along the track together.  Readings M1-M10 of DESIGN.md sec. 14.
//
//   cells      the mesh cells ARE the track macrocells (mx x my x mz sites); side 0 = trailing mesh (lower x), 1 = leading
//   state      unit direction m per cell (0 = empty cell), fp32 SoA [3][n0 + n1]
//   field      B = (2 A_0 m_e / M_S^0) lap(m) + (2 K_0 m_e^2 / M_S^0)(m.e)e + s B_app     Eq. (4), (5) with the
//              temperature scalings A = A_0 m_e^2, K = K_0 m_e^3, M_S = M_S^0 m_e, 6-neighbour stencil,
//              no exchange between different grains
//   dynamics   dm/dt = -gamma/(1+alpha^2) [m x B + alpha m x (m x B)], alpha = lambda (1 - T/3T_C); classical
//              RK4, one step of `every` * dt per `every` Heun steps, boundary data held in between
//   coupling   mesh -> atoms: the missing x neighbours of the first / last atomistic plane are the mesh directions
//              (P:60-62), handed to the Heun kernels as one extra field array per boundary plane ("edge field":
//              sum_j J_ij m_cell(j) / mu_s, constant while the mesh directions are held);
//              atoms -> mesh: the Laplacian's missing neighbour is the direction of the average atomistic spin in the
//              stencil cell; the far ends see the frozen track
//   shift      by whole cells: trailing mesh -> track, outgoing atoms -> trailing mesh by Eq. (6), leading mesh ->
//              incoming atoms by the cone thermalisation about m with magnitude m_e, track -> leading mesh
//
// The meshes are a few thousand cells: every kernel here is latency-bound and runs once per `every` Heun steps; the
// only thing the hot path pays is one predicated 128-bit load per component on the two boundary planes.
#include <cmath>
#include <cstring>
#include <new>

#include "asd_internal.cuh"

namespace asd {

struct MmPlan {
  int32_t mcx[2] = {0, 0};
  int32_t every = 1;
  int64_t age = 0;
  int32_t ncol = 0;                 // ncy * ncz: cells of one cell column plane
  int32_t n[2] = {0, 0}, ntot = 0;  // cells per side, both
  float pref[3] = {0, 0, 0};        // 2 A_0,a / (M_S^0 d_a^2), Tesla
  float mu_s = 0.f, lambda = 0.f;
  double gamma = 0.0, dt = 0.0;
  // device (caller's workspace)
  float *m = nullptr, *ya = nullptr, *yb = nullptr, *acc = nullptr;   // [3][ntot]
  float *T = nullptr, *B = nullptr;                                   // [ntot], [3][ntot]
  float *me = nullptr, *alpha = nullptr;                              // [ntot]
  int32_t* cell_grain = nullptr;                                      // [ncx*ncy]
  float* Kfac = nullptr;                                              // [G]: 2 K_0 / M_S^0, Tesla
  double* Tc = nullptr;                                               // [G]
  float* bnd = nullptr;       // [4][3][ncol]: side 0 low (track), side 0 high (atoms), side 1 low (atoms), side 1 high (track)
  float* ghost = nullptr;     // [2][3][ncol]: mesh directions next to the atoms (held)
  float* edgeB = nullptr;     // [2][3][nz*nyp]: what the meshes add to the field of atomistic planes 0 and nx-1
  float* newcols = nullptr;   // [3][maxpc*ncol] shift scratch
  float* frames = nullptr;    // [maxpc*ncol*12] cone frames of the leading mesh's outgoing columns
  float* stage = nullptr;     // host uploads land here: [4][max(n0, n1)]
  int32_t maxpc = 0;
  // m_e and alpha depend on T, B_app, the field scale and the grain under each cell: recomputed (fp64 bisection, the
  // costliest mesh kernel) only when one of those has changed since the last time
  bool params_dirty = true;
  float params_scale = 0.f;
};

namespace {

inline unsigned nblocks(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

struct MmGeom {
  int32_t mcx0, mcx1, ncy, ncz, ncol, n0, ntot;
  int32_t nx, ny, nz, nyp, lead, mx, my, mz;
  int64_t cx0[2];                   // global x index of each mesh's first cell column
  int64_t ncx;
};

__device__ __forceinline__ void cell_of(const MmGeom& g, int q, int& side, int& a, int& b, int& c) {
  side = q >= g.n0;
  const int r = side ? q - g.n0 : q;
  a = r / g.ncol;
  const int t = r - a * g.ncol;
  b = t / g.ncz; c = t - b * g.ncz;
}
__device__ __forceinline__ int32_t grain_at(const MmGeom& g, const int32_t* cell_grain, int64_t cx, int b) {
  if (cx < 0 || cx >= g.ncx || b < 0 || b >= g.ncy) return -1;
  return cell_grain[cx * g.ncy + b];
}

// Langevin function coth x - 1/x and the largest root of m = B(beta m + h), both in fp64 (set-up arithmetic).
__device__ double langevin_d(double x) {
  if (fabs(x) < 1e-3) return x / 3.0 - x * x * x / 45.0 + 2.0 * x * x * x * x * x / 945.0;
  return 1.0 / tanh(x) - 1.0 / x;
}

// m_e(T) and alpha(T) per cell.  B_ext = |s B_app| of the cell.
__global__ void mm_params_kernel(MmGeom g, const float* __restrict__ T, const float* __restrict__ B,
                                 const int32_t* __restrict__ cell_grain, const double* __restrict__ Tc, float scale,
                                 double mu_s, double lambda, float* __restrict__ me, float* __restrict__ alpha) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= g.ntot) return;
  int side, a, b, c;
  cell_of(g, q, side, a, b, c);
  const int32_t gr = grain_at(g, cell_grain, g.cx0[side] + a, b);
  if (gr < 0) { me[q] = 0.f; alpha[q] = 0.f; return; }
  const double Tq = T[q], tc = Tc[gr];
  const double bx = B[q], by = B[g.ntot + q], bz = B[2 * g.ntot + q];
  const double Bext = fabs((double)scale) * sqrt(bx * bx + by * by + bz * bz);
  double mev = 1.0;
  if (Tq > 0.0) {
    const double beta = 3.0 * tc / Tq, h = mu_s * Bext / (kBoltzmann * Tq);
    double lo = (h > 0.0) ? 0.0 : 1e-9, hi = 1.0;
    if (!(langevin_d(beta * lo + h) - lo > 0.0)) mev = 0.0;
    else {
      for (int it = 0; it < 100; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (langevin_d(beta * mid + h) - mid > 0.0) lo = mid; else hi = mid;
      }
      mev = 0.5 * (lo + hi);
    }
  }
  me[q] = (float)mev;
  alpha[q] = (float)(lambda * (1.0 - fmin(Tq, tc) / (3.0 * tc)));
}

// direction of the frozen track in cell t: what the window has written there, else what lies ahead
__device__ bool track_dir(const double* out_sum, const long long* out_cnt, const float* init_mean, int64_t t, float n[3]) {
  double v0, v1, v2;
  if (out_cnt[t] > 0) { v0 = out_sum[3 * t]; v1 = out_sum[3 * t + 1]; v2 = out_sum[3 * t + 2]; }
  else { v0 = init_mean[3 * t]; v1 = init_mean[3 * t + 1]; v2 = init_mean[3 * t + 2]; }
  const double vn = sqrt(v0 * v0 + v1 * v1 + v2 * v2);
  if (!(vn > 0.0)) return false;
  n[0] = (float)(v0 / vn); n[1] = (float)(v1 / vn); n[2] = (float)(v2 / vn);
  return true;
}

// The two-way exchange of boundary data (reading M9), one warp per (slot, b, c):
//   slots 1, 2 (atoms): direction of the sum of the atomistic spins in the stencil cell (vacant sites hold 0), fixed
//   lane order + shuffle tree in fp64; slots 0, 3 (track): direction of the frozen track cell beyond the mesh end.
//   A neighbour of another grain (or none) is stored as the zero vector.  Lane 0 also captures the mesh directions next
//   to the atoms (ghost).
__global__ void mm_exchange_kernel(MmGeom g, const float* __restrict__ sx, const float* __restrict__ sy,
                                   const float* __restrict__ sz, const float* __restrict__ m,
                                   const int32_t* __restrict__ cell_grain, const double* __restrict__ out_sum,
                                   const long long* __restrict__ out_cnt, const float* __restrict__ init_mean,
                                   int64_t cxA /* x0 / mx */, float* __restrict__ bnd, float* __restrict__ ghost) {
  const int warp = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (warp >= 4 * g.ncol) return;
  const int slot = warp / g.ncol, t = warp - slot * g.ncol;
  const int b = t / g.ncz, c = t - b * g.ncz;
  const int side = slot >> 1;
  const int mcx = side ? g.mcx1 : g.mcx0;
  const bool atoms = (slot == 1 || slot == 2);
  const int64_t cx_own = g.cx0[side] + ((slot & 1) ? mcx - 1 : 0);         // the mesh cell column at this end
  const int64_t cx_nb = (slot & 1) ? cx_own + 1 : cx_own - 1;
  const int32_t g_own = grain_at(g, cell_grain, cx_own, b);
  const bool same = g_own >= 0 && grain_at(g, cell_grain, cx_nb, b) == g_own;
  float n[3] = {0.f, 0.f, 0.f};
  if (atoms) {
    const int i_lo = side == 0 ? 0 : g.nx - g.mx;
    const int j_lo = b * g.my, nj = min((b + 1) * g.my, g.ny) - j_lo;
    const int k_lo = c * g.mz, nk = min((c + 1) * g.mz, g.nz) - k_lo;
    const int total = g.mx * nk * nj;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int q = lane; q < total; q += 32) {
      const int dj = q % nj, dk = (q / nj) % nk, di = q / (nj * nk);
      const int64_t l = g.lead + ((int64_t)(i_lo + di) * g.nz + k_lo + dk) * g.nyp + j_lo + dj;
      s0 += (double)sx[l]; s1 += (double)sy[l]; s2 += (double)sz[l];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      s0 += __shfl_down_sync(0xffffffffu, s0, off);
      s1 += __shfl_down_sync(0xffffffffu, s1, off);
      s2 += __shfl_down_sync(0xffffffffu, s2, off);
    }
    const double vn = sqrt(s0 * s0 + s1 * s1 + s2 * s2);
    if (same && vn > 0.0) { n[0] = (float)(s0 / vn); n[1] = (float)(s1 / vn); n[2] = (float)(s2 / vn); }
    (void)cxA;
  } else if (same) {
    float d[3];
    if (track_dir(out_sum, out_cnt, init_mean, (cx_nb * g.ncy + b) * g.ncz + c, d)) { n[0] = d[0]; n[1] = d[1]; n[2] = d[2]; }
  }
  if (lane == 0) {
    for (int u = 0; u < 3; ++u) bnd[(slot * 3 + u) * g.ncol + t] = n[u];
    if (atoms) {
      const int q = (side ? g.n0 : 0) + ((slot & 1) ? mcx - 1 : 0) * g.ncol + t;
      for (int u = 0; u < 3; ++u) ghost[(side * 3 + u) * g.ncol + t] = m[u * g.ntot + q];
    }
  }
}

// Edge field: what the held mesh directions add to Eq. (2) on the atomistic planes 0 (side 0) and nx-1 (side 1).
// The column table's bond bits say whether the neighbour column beyond the window edge exists in the track, is
// magnetic and belongs to the same grain.  One thread per (side, k, j); the row pads are written as zeros.
template <int LAT>
__global__ void mm_edge_kernel(MmGeom g, const uint32_t* __restrict__ col_win, const float* __restrict__ ghost,
                               float j1, float j3, float* __restrict__ edgeB) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int rowsz = g.nz * g.nyp;
  if (t >= 2 * rowsz) return;
  const int side = t / rowsz, r = t - side * rowsz;
  const int k = r / g.nyp, j = r - k * g.nyp;
  float B[3] = {0.f, 0.f, 0.f};
  if (j < g.ny) {
    const uint32_t cv = col_win[(int64_t)(side == 0 ? 0 : g.nx - 1) * g.ny + j];
    const uint32_t bX = side == 0 ? BOND_XM : BOND_XP, bP = side == 0 ? BOND_XMYP : BOND_XPYP,
                   bM = side == 0 ? BOND_XMYM : BOND_XPYM;
    const int cz = k / g.mz;
    const float* gh = ghost + side * 3 * g.ncol;
    if (cv & bX) {
      const int q = (j / g.my) * g.ncz + cz;
      for (int u = 0; u < 3; ++u) B[u] = fmaf(j1, gh[u * g.ncol + q], B[u]);
    }
    if (LAT == 1) {
      if (cv & bP) { const int q = ((j + 1) / g.my) * g.ncz + cz; for (int u = 0; u < 3; ++u) B[u] = fmaf(j3, gh[u * g.ncol + q], B[u]); }
      if (cv & bM) { const int q = ((j - 1) / g.my) * g.ncz + cz; for (int u = 0; u < 3; ++u) B[u] = fmaf(j3, gh[u * g.ncol + q], B[u]); }
    }
  }
  for (int u = 0; u < 3; ++u) edgeB[(side * 3 + u) * rowsz + r] = B[u];
}

struct MmStep {
  const float *m, *yin; float *yout, *acc;
  const float *me, *alpha, *Bapp, *bnd;
  const int32_t* cell_grain;
  const float4* grain;          // (e, 2 k_u/mu_s) per grain id + 1: the easy axes
  const float* Kfac;
  float pref[3];
  float scale, hg;              // hg = h * gamma
};

// One RK4 stage for every cell of both meshes (reading M7).  STAGE 0: k1 from m; 1, 2: k2, k3 from the stage state;
// 3: k4 and the update m <- normalise(m + (k1 + 2 k2 + 2 k3 + k4) / 6).  k carries the factor h.
template <int STAGE>
__global__ void mm_rk4_kernel(MmGeom g, MmStep s) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= g.ntot) return;
  int side, a, b, c;
  cell_of(g, q, side, a, b, c);
  const int nt = g.ntot;
  const float* Y = (STAGE == 0) ? s.m : s.yin;
  const float y[3] = {Y[q], Y[nt + q], Y[2 * nt + q]};
  const int mcx = side ? g.mcx1 : g.mcx0;
  const int32_t gr = grain_at(g, s.cell_grain, g.cx0[side] + a, b);
  const float mev = s.me[q];
  float k[3] = {0.f, 0.f, 0.f};
  if (gr >= 0 && mev > 0.f) {
    float L[3] = {0.f, 0.f, 0.f};                       // sum_a pref_a (m_n - m)
    auto add = [&](float n0, float n1, float n2, float pa) {
      L[0] = fmaf(pa, n0 - y[0], L[0]); L[1] = fmaf(pa, n1 - y[1], L[1]); L[2] = fmaf(pa, n2 - y[2], L[2]);
    };
    // x: inside the mesh, or the boundary slot of this end (a zero vector = no neighbour)
#pragma unroll
    for (int dir = 0; dir < 2; ++dir) {
      const int a2 = a + (dir ? 1 : -1);
      if (a2 >= 0 && a2 < mcx) {
        if (grain_at(g, s.cell_grain, g.cx0[side] + a2, b) == gr) {
          const int q2 = q + (dir ? g.ncol : -g.ncol);
          add(Y[q2], Y[nt + q2], Y[2 * nt + q2], s.pref[0]);
        }
      } else {
        const float* bp = s.bnd + (side * 2 + dir) * 3 * g.ncol + (b * g.ncz + c);
        const float n0 = bp[0], n1 = bp[g.ncol], n2 = bp[2 * g.ncol];
        if (n0 != 0.f || n1 != 0.f || n2 != 0.f) add(n0, n1, n2, s.pref[0]);
      }
    }
#pragma unroll
    for (int dir = 0; dir < 2; ++dir) {                 // y: the next cell column across the track
      const int b2 = b + (dir ? 1 : -1);
      if (b2 >= 0 && b2 < g.ncy && grain_at(g, s.cell_grain, g.cx0[side] + a, b2) == gr) {
        const int q2 = q + (dir ? g.ncz : -g.ncz);
        add(Y[q2], Y[nt + q2], Y[2 * nt + q2], s.pref[1]);
      }
    }
    if (c > 0) add(Y[q - 1], Y[nt + q - 1], Y[2 * nt + q - 1], s.pref[2]);            // z: same column, same grain
    if (c + 1 < g.ncz) add(Y[q + 1], Y[nt + q + 1], Y[2 * nt + q + 1], s.pref[2]);
    const float4 e = __ldg(s.grain + gr + 1);
    const float ca = s.Kfac[gr] * mev * mev * fmaf(y[0], e.x, fmaf(y[1], e.y, y[2] * e.z));
    const float B0 = fmaf(mev, L[0], fmaf(ca, e.x, s.scale * s.Bapp[q]));
    const float B1 = fmaf(mev, L[1], fmaf(ca, e.y, s.scale * s.Bapp[nt + q]));
    const float B2 = fmaf(mev, L[2], fmaf(ca, e.z, s.scale * s.Bapp[2 * nt + q]));
    const float a0 = y[1] * B2 - y[2] * B1, a1 = y[2] * B0 - y[0] * B2, a2 = y[0] * B1 - y[1] * B0;
    const float b0 = y[1] * a2 - y[2] * a1, b1 = y[2] * a0 - y[0] * a2, b2 = y[0] * a1 - y[1] * a0;
    const float al = s.alpha[q], cf = -s.hg / (1.0f + al * al);
    k[0] = cf * fmaf(al, b0, a0); k[1] = cf * fmaf(al, b1, a1); k[2] = cf * fmaf(al, b2, a2);
  }
  const float m0[3] = {s.m[q], s.m[nt + q], s.m[2 * nt + q]};
  if (STAGE == 0) {
    for (int u = 0; u < 3; ++u) { s.acc[u * nt + q] = k[u]; s.yout[u * nt + q] = fmaf(0.5f, k[u], m0[u]); }
  } else if (STAGE == 1) {
    for (int u = 0; u < 3; ++u) { s.acc[u * nt + q] += 2.0f * k[u]; s.yout[u * nt + q] = fmaf(0.5f, k[u], m0[u]); }
  } else if (STAGE == 2) {
    for (int u = 0; u < 3; ++u) { s.acc[u * nt + q] += 2.0f * k[u]; s.yout[u * nt + q] = m0[u] + k[u]; }
  } else {
    float v[3];
    for (int u = 0; u < 3; ++u) v[u] = fmaf(1.0f / 6.0f, s.acc[u * nt + q] + k[u], m0[u]);
    const float n2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    const float inv = n2 > 0.f ? 1.0f / sqrtf(n2) : 0.f;
    for (int u = 0; u < 3; ++u) s.yout[u * nt + q] = v[u] * inv;       // yout = m for this stage
  }
}

// Initial state: the direction of the track the meshes lie over; empty cells 0.
__global__ void mm_init_kernel(MmGeom g, const int32_t* __restrict__ cell_grain, const double* __restrict__ out_sum,
                               const long long* __restrict__ out_cnt, const float* __restrict__ init_mean,
                               float* __restrict__ m) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= g.ntot) return;
  int side, a, b, c;
  cell_of(g, q, side, a, b, c);
  float n[3] = {0.f, 0.f, 0.f};
  if (grain_at(g, cell_grain, g.cx0[side] + a, b) >= 0) {
    n[2] = 1.f;
    float d[3];
    if (track_dir(out_sum, out_cnt, init_mean, ((g.cx0[side] + a) * g.ncy + b) * g.ncz + c, d)) { n[0] = d[0]; n[1] = d[1]; n[2] = d[2]; }
  }
  for (int u = 0; u < 3; ++u) m[u * g.ntot + q] = n[u];
}

// ---- shift by pc whole cells (reading M10) ----
// 1. trailing mesh columns a < pc -> track: M / M_S^0 = m_e m on the magnetic sites of the cell.
// (side 0, pc columns at a shift; all columns of either mesh at the end of a pass)
__global__ void mm_out_to_track_kernel(MmGeom g, int side, int pc, const float* __restrict__ m, const float* __restrict__ me,
                                       const int32_t* __restrict__ cell_grain, const uint32_t* __restrict__ col_track,
                                       int64_t track_nx, double* __restrict__ out_sum, long long* __restrict__ out_cnt) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= pc * g.ncol) return;
  const int a = r / g.ncol, t = r - a * g.ncol, b = t / g.ncz, c = t - b * g.ncz;
  const int q = (side ? g.n0 : 0) + r;
  const int64_t cx = g.cx0[side] + a;
  if (grain_at(g, cell_grain, cx, b) < 0) return;
  long long n = 0;
  const int kext = min((c + 1) * g.mz, g.nz) - c * g.mz;
  for (int64_t gx = cx * g.mx; gx < min((cx + 1) * (int64_t)g.mx, track_nx); ++gx)
    for (int j = b * g.my; j < min((b + 1) * g.my, g.ny); ++j)
      if ((col_track[gx * g.ny + j] & 0xFFFFu) != 0u) n += kext;
  const int64_t tc = (cx * g.ncy + b) * g.ncz + c;
  const double w = (double)me[q] * (double)n;
  out_sum[3 * tc] += w * (double)m[q]; out_sum[3 * tc + 1] += w * (double)m[g.ntot + q];
  out_sum[3 * tc + 2] += w * (double)m[2 * g.ntot + q];
  out_cnt[tc] += n;
}
// 2. new trailing-mesh columns: direction of the Eq. (6) sum over the outgoing atomistic cell; one warp per cell.
__global__ void mm_new_trailing_kernel(MmGeom g, int pc, const float* __restrict__ sx, const float* __restrict__ sy,
                                       const float* __restrict__ sz, const int32_t* __restrict__ cell_grain, int64_t cxA,
                                       float* __restrict__ newcols) {
  const int warp = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (warp >= pc * g.ncol) return;
  const int a = warp / g.ncol, t = warp - a * g.ncol, b = t / g.ncz, c = t - b * g.ncz;
  const int j_lo = b * g.my, nj = min((b + 1) * g.my, g.ny) - j_lo;
  const int k_lo = c * g.mz, nk = min((c + 1) * g.mz, g.nz) - k_lo;
  const int total = g.mx * nk * nj;
  double s0 = 0.0, s1 = 0.0, s2 = 0.0;
  for (int q = lane; q < total; q += 32) {
    const int dj = q % nj, dk = (q / nj) % nk, di = q / (nj * nk);
    const int64_t l = g.lead + ((int64_t)(a * g.mx + di) * g.nz + k_lo + dk) * g.nyp + j_lo + dj;
    s0 += (double)sx[l]; s1 += (double)sy[l]; s2 += (double)sz[l];
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    s0 += __shfl_down_sync(0xffffffffu, s0, off);
    s1 += __shfl_down_sync(0xffffffffu, s1, off);
    s2 += __shfl_down_sync(0xffffffffu, s2, off);
  }
  if (lane == 0) {
    float n[3] = {0.f, 0.f, 0.f};
    if (grain_at(g, cell_grain, cxA + a, b) >= 0) {
      const double vn = sqrt(s0 * s0 + s1 * s1 + s2 * s2);
      if (vn > 0.0) { n[0] = (float)(s0 / vn); n[1] = (float)(s1 / vn); n[2] = (float)(s2 / vn); } else n[2] = 1.f;
    }
    const int stride = pc * g.ncol;
    for (int u = 0; u < 3; ++u) newcols[u * stride + warp] = n[u];
  }
}
// 3. cone frames of the leading mesh's first pc columns: v = m_e m -> theta_max, (n, e1, e2) as cell_frames_kernel does
__global__ void mm_frames_kernel(MmGeom g, int pc, const float* __restrict__ m, const float* __restrict__ me,
                                 float* __restrict__ frames) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= pc * g.ncol) return;
  const int q = g.n0 + t;
  const double mev = me[q];
  const double v0 = mev * m[q], v1 = mev * m[g.ntot + q], v2 = mev * m[2 * g.ntot + q];
  const double vn = sqrt(v0 * v0 + v1 * v1 + v2 * v2);
  const double mm_ = fmin(1.0, vn);
  double n0 = 0.0, n1 = 0.0, n2 = 1.0;
  if (vn > 0.0) { n0 = v0 / vn; n1 = v1 / vn; n2 = v2 / vn; }
  double a0, a1, a2;
  if (fabs(n0) > 0.9) { a0 = -n2; a1 = 0.0; a2 = n0; } else { a0 = 0.0; a1 = n2; a2 = -n1; }
  const double an = sqrt(a0 * a0 + a1 * a1 + a2 * a2);
  a0 /= an; a1 /= an; a2 /= an;
  const double b0 = n1 * a2 - n2 * a1, b1 = n2 * a0 - n0 * a2, b2 = n0 * a1 - n1 * a0;
  double th;
  if (mm_ >= 1.0) th = 0.0;
  else if (mm_ <= 0.0) th = 3.14159265358979323846;
  else {
    double lo = 0.0, hi = 3.14159265358979323846;
    for (int it = 0; it < 60; ++it) { const double mid = 0.5 * (lo + hi); if (sin(mid) > mm_ * mid) lo = mid; else hi = mid; }
    th = 0.5 * (lo + hi);
  }
  float* f = frames + 12 * t;
  f[0] = (float)th; f[1] = (float)n0; f[2] = (float)n1; f[3] = (float)n2;
  f[4] = (float)a0; f[5] = (float)a1; f[6] = (float)a2; f[7] = (float)b0; f[8] = (float)b1; f[9] = (float)b2;
  f[10] = 0.f; f[11] = 0.f;
}
// 4. both meshes move by pc columns into `dst`; trailing mesh's new columns = newcols, leading mesh's = the track ahead
__global__ void mm_move_kernel(MmGeom g, int pc, const float* __restrict__ m, const float* __restrict__ newcols,
                               const int32_t* __restrict__ cell_grain, const float* __restrict__ init_mean,
                               float* __restrict__ dst) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= g.ntot) return;
  int side, a, b, c;
  cell_of(g, q, side, a, b, c);
  const int mcx = side ? g.mcx1 : g.mcx0;
  float n[3];
  if (a + pc < mcx) {
    for (int u = 0; u < 3; ++u) n[u] = m[u * g.ntot + q + pc * g.ncol];
  } else if (side == 0) {
    const int t = (a - (mcx - pc)) * g.ncol + b * g.ncz + c, stride = pc * g.ncol;
    for (int u = 0; u < 3; ++u) n[u] = newcols[u * stride + t];
  } else {
    n[0] = n[1] = n[2] = 0.f;
    const int64_t cx = g.cx0[1] + pc + a;                 // its global cell column AFTER the move
    if (grain_at(g, cell_grain, cx, b) >= 0) {
      const int64_t t = (cx * g.ncy + b) * g.ncz + c;
      const double v0 = init_mean[3 * t], v1 = init_mean[3 * t + 1], v2 = init_mean[3 * t + 2];
      const double vn = sqrt(v0 * v0 + v1 * v1 + v2 * v2);
      if (vn > 0.0) { n[0] = (float)(v0 / vn); n[1] = (float)(v1 / vn); n[2] = (float)(v2 / vn); } else n[2] = 1.f;
    }
  }
  for (int u = 0; u < 3; ++u) dst[u * g.ntot + q] = n[u];
}

// host AoS [cells][3] <-> device SoA of one side
__global__ void mm_aos_to_soa_kernel(MmGeom g, int side, const float* __restrict__ src, const int32_t* __restrict__ cell_grain,
                                     float* __restrict__ m) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  const int n = side ? g.ntot - g.n0 : g.n0;
  if (r >= n) return;
  const int q = (side ? g.n0 : 0) + r;
  const int a = r / g.ncol, b = (r - a * g.ncol) / g.ncz;
  const bool full = grain_at(g, cell_grain, g.cx0[side] + a, b) >= 0;
  for (int u = 0; u < 3; ++u) m[u * g.ntot + q] = full ? src[3 * r + u] : 0.f;
}
__global__ void mm_soa_to_aos_kernel(MmGeom g, int side, const float* __restrict__ m, float* __restrict__ dst) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  const int n = side ? g.ntot - g.n0 : g.n0;
  if (r >= n) return;
  const int q = (side ? g.n0 : 0) + r;
  for (int u = 0; u < 3; ++u) dst[3 * r + u] = m[u * g.ntot + q];
}

MmGeom geom(const Ctx& c) {
  const MmPlan& P = *c.mm;
  MmGeom g;
  g.mcx0 = P.mcx[0]; g.mcx1 = P.mcx[1]; g.ncy = (int32_t)c.ncy; g.ncz = (int32_t)c.ncz; g.ncol = P.ncol;
  g.n0 = P.n[0]; g.ntot = P.ntot;
  g.nx = c.d.nx; g.ny = c.d.ny; g.nz = c.d.nz; g.nyp = c.nyp; g.lead = c.lead;
  g.mx = c.d.macro[0]; g.my = c.d.macro[1]; g.mz = c.d.macro[2];
  g.cx0[0] = c.x0 / g.mx - P.mcx[0]; g.cx0[1] = (c.x0 + c.d.nx) / g.mx;
  g.ncx = c.ncx;
  return g;
}

struct MmLayout { size_t m, ya, yb, acc, T, B, me, alpha, cell_grain, Kfac, Tc, bnd, ghost, edgeB, newcols, frames, stage, total; };
MmLayout layout(const Ctx& c, const int32_t mcx[2]) {
  MmLayout L;
  const size_t ncol = (size_t)(c.ncy * c.ncz), ntot = ncol * (size_t)(mcx[0] + mcx[1]);
  const size_t maxpc = (size_t)(mcx[0] < mcx[1] ? mcx[0] : mcx[1]);
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes, 256); return o; };
  L.m = take(12 * ntot); L.ya = take(12 * ntot); L.yb = take(12 * ntot); L.acc = take(12 * ntot);
  L.T = take(4 * ntot); L.B = take(12 * ntot); L.me = take(4 * ntot); L.alpha = take(4 * ntot);
  L.cell_grain = take(4 * (size_t)(c.ncx * c.ncy));
  L.Kfac = take(4 * (size_t)c.d.n_grains); L.Tc = take(8 * (size_t)c.d.n_grains);
  L.bnd = take(4 * 12 * ncol); L.ghost = take(4 * 6 * ncol);
  L.edgeB = take(4 * 6 * (size_t)c.d.nz * (size_t)c.nyp);
  L.newcols = take(12 * maxpc * ncol); L.frames = take(48 * maxpc * ncol);
  const size_t nmax = ncol * (size_t)(mcx[0] > mcx[1] ? mcx[0] : mcx[1]);
  L.stage = take(16 * nmax);
  L.total = off;
  return L;
}

asd_status launch_params(Ctx& c) {
  MmPlan& P = *c.mm;
  mm_params_kernel<<<nblocks(P.ntot, 128), 128, 0, c.stream>>>(geom(c), P.T, P.B, P.cell_grain, P.Tc, c.scale,
                                                             c.d.mu_s, c.d.lambda, P.me, P.alpha);
  ASD_LAUNCH_CHECK(c, "mm_params");
  P.params_dirty = false; P.params_scale = c.scale;
  return ASD_OK;
}

asd_status launch_exchange(Ctx& c) {
  MmPlan& P = *c.mm;
  const MmGeom g = geom(c);
  const Vec3Ptr S = c.S();
  mm_exchange_kernel<<<nblocks((int64_t)4 * P.ncol * 32, 128), 128, 0, c.stream>>>(
      g, S.x, S.y, S.z, P.m, P.cell_grain, c.out_sum, c.out_cnt, c.init_mean, c.x0 / g.mx, P.bnd, P.ghost);
  ASD_LAUNCH_CHECK(c, "mm_exchange");
  const float j1 = (float)(c.d.J[0] / c.d.mu_s), j3 = (float)(c.d.J[2] / c.d.mu_s);
  const int n = 2 * c.d.nz * c.nyp;
  if (c.d.lattice == ASD_SC) mm_edge_kernel<0><<<nblocks(n, 128), 128, 0, c.stream>>>(g, c.col_win(), P.ghost, j1, j3, P.edgeB);
  else mm_edge_kernel<1><<<nblocks(n, 128), 128, 0, c.stream>>>(g, c.col_win(), P.ghost, j1, j3, P.edgeB);
  ASD_LAUNCH_CHECK(c, "mm_edge");
  return ASD_OK;
}

asd_status launch_rk4(Ctx& c, double h) {
  MmPlan& P = *c.mm;
  const MmGeom g = geom(c);
  MmStep s;
  s.m = P.m; s.acc = P.acc; s.me = P.me; s.alpha = P.alpha; s.Bapp = P.B; s.bnd = P.bnd;
  s.cell_grain = P.cell_grain; s.grain = c.grain; s.Kfac = P.Kfac;
  for (int a = 0; a < 3; ++a) s.pref[a] = P.pref[a];
  s.scale = c.scale; s.hg = (float)(h * c.gamma);
  const unsigned nb = nblocks(P.ntot, 128);
  s.yin = nullptr; s.yout = P.ya;
  mm_rk4_kernel<0><<<nb, 128, 0, c.stream>>>(g, s); ASD_LAUNCH_CHECK(c, "mm_rk4 k1");
  s.yin = P.ya; s.yout = P.yb;
  mm_rk4_kernel<1><<<nb, 128, 0, c.stream>>>(g, s); ASD_LAUNCH_CHECK(c, "mm_rk4 k2");
  s.yin = P.yb; s.yout = P.ya;
  mm_rk4_kernel<2><<<nb, 128, 0, c.stream>>>(g, s); ASD_LAUNCH_CHECK(c, "mm_rk4 k3");
  s.yin = P.ya; s.yout = P.m;                            // stage 3 reads its neighbours from ya and writes m in place
  mm_rk4_kernel<3><<<nb, 128, 0, c.stream>>>(g, s); ASD_LAUNCH_CHECK(c, "mm_rk4 k4");
  return ASD_OK;
}

}  // namespace

const float* mm_edge_field(const Ctx& c) { return c.mm ? c.mm->edgeB : (c.tex_on ? c.tex_edgeB : nullptr); }

// ---- window ends exchange coupled to the frozen track (reading E1), for a purely atomistic window ----
namespace {
// ghost[side][u][b*ncz + c] = direction of the frozen track in the macrocell that holds the plane just beyond the window
// end (side 0: plane x0 - 1; side 1: plane x0 + nx); 0 where there is no track or no direction.
__global__ void track_ghost_kernel(int ncy, int ncz, long long ncx, long long cxg0, long long cxg1,
                                   const double* __restrict__ out_sum, const long long* __restrict__ out_cnt,
                                   const float* __restrict__ init_mean, float* __restrict__ ghost) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x, ncol = ncy * ncz;
  if (t >= 2 * ncol) return;
  const int side = t / ncol, r = t - side * ncol;
  const long long cx = side ? cxg1 : cxg0;
  float n[3] = {0.f, 0.f, 0.f}, d[3];
  if (cx >= 0 && cx < ncx && track_dir(out_sum, out_cnt, init_mean, cx * ncol + r, d)) { n[0] = d[0]; n[1] = d[1]; n[2] = d[2]; }
  for (int u = 0; u < 3; ++u) ghost[(side * 3 + u) * ncol + r] = n[u];
}
}  // namespace

size_t track_exchange_workspace_bytes(const Ctx& c) {
  return align_up(sizeof(float) * 6 * (size_t)(c.ncy * c.ncz), 256) + align_up(sizeof(float) * 6 * (size_t)c.d.nz * (size_t)c.nyp, 256);
}

asd_status track_exchange_refresh(Ctx& c) {
  if (!c.tex_on || c.mm) return ASD_OK;                   // the meshes of a multiscale window take over the ends
  const int mx = c.d.macro[0], ncol = (int)(c.ncy * c.ncz);
  const long long cxg0 = c.x0 > 0 ? (c.x0 - 1) / mx : -1, cxg1 = (c.x0 + c.d.nx < c.d.track_nx) ? (c.x0 + c.d.nx) / mx : -1;
  track_ghost_kernel<<<nblocks(2 * ncol, 128), 128, 0, c.stream>>>((int)c.ncy, (int)c.ncz, (long long)c.ncx, cxg0, cxg1,
                                                                  c.out_sum, c.out_cnt, c.init_mean, c.tex_ghost);
  ASD_LAUNCH_CHECK(c, "track_ghost");
  MmGeom g = {};
  g.ncy = (int32_t)c.ncy; g.ncz = (int32_t)c.ncz; g.ncol = ncol;
  g.nx = c.d.nx; g.ny = c.d.ny; g.nz = c.d.nz; g.nyp = c.nyp; g.lead = c.lead;
  g.mx = mx; g.my = c.d.macro[1]; g.mz = c.d.macro[2];
  const float j1 = (float)(c.d.J[0] / c.d.mu_s), j3 = (float)(c.d.J[2] / c.d.mu_s);
  const int n = 2 * c.d.nz * c.nyp;
  if (c.d.lattice == ASD_SC) mm_edge_kernel<0><<<nblocks(n, 128), 128, 0, c.stream>>>(g, c.col_win(), c.tex_ghost, j1, j3, c.tex_edgeB);
  else mm_edge_kernel<1><<<nblocks(n, 128), 128, 0, c.stream>>>(g, c.col_win(), c.tex_ghost, j1, j3, c.tex_edgeB);
  ASD_LAUNCH_CHECK(c, "track_edge");
  return ASD_OK;
}

asd_status track_exchange_enable(Ctx& c, int on, void* ws, size_t bytes) {
  if (!on) { c.tex_on = false; return ASD_OK; }
  if (bytes < track_exchange_workspace_bytes(c)) { std::snprintf(c.err, sizeof(c.err), "asd_enable_track_exchange: workspace too small"); return ASD_ENOMEM; }
  c.tex_ghost = (float*)ws;
  c.tex_edgeB = (float*)((char*)ws + align_up(sizeof(float) * 6 * (size_t)(c.ncy * c.ncz), 256));
  c.tex_on = true;
  return track_exchange_refresh(c);
}

// Called before every Heun step (reading M9): every `every`-th step the meshes and the atoms trade boundary data (from
// the configurations at that instant) and the meshes advance by one RK4 step of every * dt.
asd_status mm_before_step(Ctx& c) {
  MmPlan& P = *c.mm;
  if (P.age % P.every == 0) {
    asd_status st = launch_exchange(c);
    if (st == ASD_OK && (P.params_dirty || P.params_scale != c.scale)) st = launch_params(c);
    if (st == ASD_OK) st = launch_rk4(c, (double)P.every * c.d.dt);
    if (st != ASD_OK) return st;
  }
  P.age += 1;
  return ASD_OK;
}

void mm_restart_cadence(Ctx& c) { if (c.mm) c.mm->age = 0; }

size_t mm_workspace_bytes(const Ctx& c, const int32_t mcx[2]) { return layout(c, mcx).total; }

void mm_free(Ctx& c) { delete c.mm; c.mm = nullptr; }

asd_status mm_enable(Ctx& c, const asd_mm_desc& d, void* ws, size_t bytes) {
  const MmLayout L = layout(c, d.mcx);
  if (bytes < L.total) { std::snprintf(c.err, sizeof(c.err), "asd_mm_enable: workspace too small"); return ASD_ENOMEM; }
  MmPlan* P = c.mm ? c.mm : new (std::nothrow) MmPlan();
  if (!P) return ASD_ENOMEM;
  c.mm = P;
  P->mcx[0] = d.mcx[0]; P->mcx[1] = d.mcx[1]; P->every = d.every; P->age = 0;
  P->ncol = (int32_t)(c.ncy * c.ncz);
  P->n[0] = P->ncol * d.mcx[0]; P->n[1] = P->ncol * d.mcx[1]; P->ntot = P->n[0] + P->n[1];
  P->maxpc = d.mcx[0] < d.mcx[1] ? d.mcx[0] : d.mcx[1];
  for (int a = 0; a < 3; ++a) {
    const double cell = c.d.macro[a] * d.spacing_m[a];
    P->pref[a] = (float)(2.0 * d.A0[a] / (d.Ms0 * cell * cell));
  }
  char* base = (char*)ws;
  P->m = (float*)(base + L.m); P->ya = (float*)(base + L.ya); P->yb = (float*)(base + L.yb); P->acc = (float*)(base + L.acc);
  P->T = (float*)(base + L.T); P->B = (float*)(base + L.B); P->me = (float*)(base + L.me); P->alpha = (float*)(base + L.alpha);
  P->cell_grain = (int32_t*)(base + L.cell_grain); P->Kfac = (float*)(base + L.Kfac); P->Tc = (double*)(base + L.Tc);
  P->bnd = (float*)(base + L.bnd); P->ghost = (float*)(base + L.ghost); P->edgeB = (float*)(base + L.edgeB);
  P->newcols = (float*)(base + L.newcols); P->frames = (float*)(base + L.frames); P->stage = (float*)(base + L.stage);
  ASD_CUDA_TRY(c, cudaMemsetAsync(ws, 0, L.total, c.stream));
  ASD_CUDA_TRY(c, cudaMemcpyAsync(P->cell_grain, d.cell_grain, 4 * (size_t)(c.ncx * c.ncy), cudaMemcpyHostToDevice, c.stream));
  ASD_CUDA_TRY(c, cudaMemcpyAsync(P->Tc, d.Tc, 8 * (size_t)c.d.n_grains, cudaMemcpyHostToDevice, c.stream));
  {
    float* kf = nullptr;
    ASD_CUDA_TRY(c, cudaMallocHost(&kf, 4 * (size_t)c.d.n_grains));
    for (int g = 0; g < c.d.n_grains; ++g) kf[g] = (float)(2.0 * d.K0[g] / d.Ms0);
    cudaError_t e = cudaMemcpyAsync(P->Kfac, kf, 4 * (size_t)c.d.n_grains, cudaMemcpyHostToDevice, c.stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c.stream);     // also covers the pageable copies above
    cudaFreeHost(kf);
    if (e != cudaSuccess) return fail_cuda(c, e, "asd_mm_enable upload");
  }
  mm_init_kernel<<<nblocks(P->ntot, 128), 128, 0, c.stream>>>(geom(c), P->cell_grain, c.out_sum, c.out_cnt, c.init_mean, P->m);
  ASD_LAUNCH_CHECK(c, "mm_init");
  return launch_params(c);
}

asd_status mm_set_fields_host(Ctx& c, int side, const float* T, const float* Bx, const float* By, const float* Bz) {
  MmPlan& P = *c.mm;
  const size_t n = (size_t)P.n[side], off = side ? (size_t)P.n[0] : 0;
  const float* src[4] = {T, Bx, By, Bz};
  float* dst[4] = {P.T + off, P.B + off, P.B + P.ntot + off, P.B + 2 * (size_t)P.ntot + off};
  for (int a = 0; a < 4; ++a)
    if (src[a]) ASD_CUDA_TRY(c, cudaMemcpyAsync(dst[a], src[a], 4 * n, cudaMemcpyHostToDevice, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));       // the caller's arrays may be pageable temporaries
  return launch_params(c);
}

asd_status mm_set_m_host(Ctx& c, int side, const float* m) {
  MmPlan& P = *c.mm;
  ASD_CUDA_TRY(c, cudaMemcpyAsync(P.stage, m, 12 * (size_t)P.n[side], cudaMemcpyHostToDevice, c.stream));
  mm_aos_to_soa_kernel<<<nblocks(P.n[side], 128), 128, 0, c.stream>>>(geom(c), side, P.stage, P.cell_grain, P.m);
  ASD_LAUNCH_CHECK(c, "mm_set_m");
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  P.age = 0;
  return ASD_OK;
}

asd_status mm_get_m_host(Ctx& c, int side, float* m) {
  MmPlan& P = *c.mm;
  mm_soa_to_aos_kernel<<<nblocks(P.n[side], 128), 128, 0, c.stream>>>(geom(c), side, P.m, P.stage);
  ASD_LAUNCH_CHECK(c, "mm_get_m");
  ASD_CUDA_TRY(c, cudaMemcpyAsync(m, P.stage, 12 * (size_t)P.n[side], cudaMemcpyDeviceToHost, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  return ASD_OK;
}

void mm_dims(const Ctx& c, int side, int64_t dims[3]) { dims[0] = c.mm->mcx[side]; dims[1] = c.ncy; dims[2] = c.ncz; }

// The mesh part of a whole-cell shift, BEFORE the atomistic planes move (launch_shift_mm in asd_shift.cu does the rest):
// trailing mesh -> track, outgoing atoms -> newcols, cone frames of the leading mesh's first pc columns.
asd_status mm_shift_prepare(Ctx& c, int pc) {
  MmPlan& P = *c.mm;
  const MmGeom g = geom(c);
  const Vec3Ptr S = c.S();
  mm_out_to_track_kernel<<<nblocks((int64_t)pc * P.ncol, 128), 128, 0, c.stream>>>(g, 0, pc, P.m, P.me, P.cell_grain, c.col,
                                                                                 c.d.track_nx, c.out_sum, c.out_cnt);
  ASD_LAUNCH_CHECK(c, "mm_out_to_track");
  mm_new_trailing_kernel<<<nblocks((int64_t)pc * P.ncol * 32, 128), 128, 0, c.stream>>>(g, pc, S.x, S.y, S.z, P.cell_grain,
                                                                                      c.x0 / g.mx, P.newcols);
  ASD_LAUNCH_CHECK(c, "mm_new_trailing");
  mm_frames_kernel<<<nblocks((int64_t)pc * P.ncol, 128), 128, 0, c.stream>>>(g, pc, P.m, P.me, P.frames);
  ASD_LAUNCH_CHECK(c, "mm_frames");
  return ASD_OK;
}
const float* mm_shift_frames(const Ctx& c) { return c.mm->frames; }

// End of a pass (reading T1'): every cell of both meshes goes to the track store.
asd_status mm_flush_to_track(Ctx& c) {
  MmPlan& P = *c.mm;
  const MmGeom g = geom(c);
  for (int side = 0; side < 2; ++side) {
    mm_out_to_track_kernel<<<nblocks(P.n[side], 128), 128, 0, c.stream>>>(g, side, P.mcx[side], P.m, P.me, P.cell_grain, c.col,
                                                                        c.d.track_nx, c.out_sum, c.out_cnt);
    ASD_LAUNCH_CHECK(c, "mm_out_to_track(all columns)");
  }
  return ASD_OK;
}
// Start of a pass (reading T2'): the meshes restart along the track they lie over at the context's (new) window origin.
asd_status mm_restart_from_track(Ctx& c) {
  MmPlan& P = *c.mm;
  mm_init_kernel<<<nblocks(P.ntot, 128), 128, 0, c.stream>>>(geom(c), P.cell_grain, c.out_sum, c.out_cnt, c.init_mean, P.m);
  ASD_LAUNCH_CHECK(c, "mm_init");
  P.age = 0;
  return launch_params(c);
}
// ... and AFTER: both meshes move by pc columns (geometry still that of the old window origin).
asd_status mm_shift_finish(Ctx& c, int pc) {
  MmPlan& P = *c.mm;
  mm_move_kernel<<<nblocks(P.ntot, 128), 128, 0, c.stream>>>(geom(c), pc, P.m, P.newcols, P.cell_grain, c.init_mean, P.ya);
  ASD_LAUNCH_CHECK(c, "mm_move");
  ASD_CUDA_TRY(c, cudaMemcpyAsync(P.m, P.ya, 12 * (size_t)P.ntot, cudaMemcpyDeviceToDevice, c.stream));
  P.age = 0;
  P.params_dirty = true;                                 // other grains now lie under the window-fixed profiles
  return ASD_OK;
}

}  // namespace asd
