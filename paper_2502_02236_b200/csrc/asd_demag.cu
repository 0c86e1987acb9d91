// asd_demag.cu -- demagnetising field of the atomistic window (Eq. (6)-(7)).
//
//   M_c = (mu_s / V) sum_{j in c} X_j                  Eq. (6): spins -> macrocell magnetisation (V = full cell volume)
//   B_c = -mu_0 sum_c' N(r_c' - r_c) M_c'               Eq. (7): convolution with the cuboid demagnetising tensor
//
// evaluated for the configuration of EVERY Heun stage (the paper recomputes it "at every iteration") over the
// track macrocells that overlap the window (open boundaries; the frozen track's stray field is not included -- callers
// add it through the per-site B arrays).  Each site then sees the field of its macrocell.
//
// Per stage, in stream order:  coarse_grain_cells (coalesced row sweeps, fixed summation order, deterministic)
//   -> cuFFT R2C of the 3 zero-padded components -> multiply_tensor (6 real-even kernels, transformed once at set-up)
//   -> cuFFT C2R -> the stage kernel adds demag_B[cell(site)] to its exchange field.
// The FFT is the one library primitive on this path (like cuBLAS for a plain GEMM); everything around it is ours.
// The tensor itself is computed on the host in fp64 at enable time.
#include <cufft.h>

#include <cmath>
#include <vector>

#include "asd_internal.cuh"

namespace asd {

struct DemagPlan {
  int dcx = 0, dcy = 0, dcz = 0;      // macrocells that can overlap the window (x: worst alignment of x0)
  int px = 0, py = 0, pz = 0, pzc = 0; // padded transform size, and pz/2 + 1
  double cell[3] = {0, 0, 0};
  float mu_over_V = 0.0f;
  float* M = nullptr;                 // [3][px][py][pz]
  cufftComplex* Mh = nullptr;         // [3][px][py][pzc]
  cufftComplex* Kh = nullptr;         // [6][px][py][pzc], includes -mu_0 / (px py pz)
  float* B = nullptr;                 // [3][px][py][pz]
  cufftHandle fwd = 0, inv = 0;
  bool plans = false;
};

namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr double kNearDiagonals = 12.0;     // beyond this many cell diagonals: point dipoles (reading D2)

// Newell, Williams and Dunlop (1993) auxiliary functions, arguments taken by absolute value (parity restored by the caller).
double aux_diag(double a, double b, double c) {       // "f": enters N_aa with a along the tensor axis
  a = std::fabs(a); b = std::fabs(b); c = std::fabs(c);
  const double r = std::sqrt(a * a + b * b + c * c);
  if (r == 0.0) return 0.0;
  double s = r * (2.0 * a * a - b * b - c * c) / 6.0;
  const double ac = std::sqrt(a * a + c * c), ab = std::sqrt(a * a + b * b);
  if (b > 0.0 && ac > 0.0) s += 0.5 * b * (c * c - a * a) * std::asinh(b / ac);
  if (c > 0.0 && ab > 0.0) s += 0.5 * c * (b * b - a * a) * std::asinh(c / ab);
  if (a > 0.0 && b > 0.0 && c > 0.0) s -= a * b * c * std::atan(b * c / (a * r));
  return s;
}
double aux_offdiag(double a, double b, double c) {    // "g": enters N_ab with (a, b) the tensor axes; odd in a and b
  const double parity = (a < 0.0 ? -1.0 : 1.0) * (b < 0.0 ? -1.0 : 1.0);
  a = std::fabs(a); b = std::fabs(b); c = std::fabs(c);
  const double r = std::sqrt(a * a + b * b + c * c);
  if (r == 0.0 || a == 0.0 || b == 0.0) return 0.0;   // every term carries a factor a b or vanishes with it
  double s = -a * b * r / 3.0;
  if (c > 0.0) s += a * b * c * std::asinh(c / std::sqrt(a * a + b * b));
  s += b * (3.0 * c * c - b * b) / 6.0 * std::asinh(a / std::sqrt(b * b + c * c));
  s += a * (3.0 * c * c - a * a) / 6.0 * std::asinh(b / std::sqrt(a * a + c * c));
  if (c > 0.0) {
    s -= c * c * c / 6.0 * std::atan(a * b / (c * r));
    s -= 0.5 * c * b * b * std::atan(a * c / (b * r));
    s -= 0.5 * c * a * a * std::atan(b * c / (a * r));
  }
  return parity * s;
}

// (Nxx, Nyy, Nzz, Nxy, Nxz, Nyz) for cell edges d and centre offset R: -1/(4 pi V) times the 27-point second difference.
void cuboid_tensor(const double d[3], const double R[3], double N[6]) {
  const double V = d[0] * d[1] * d[2];
  const double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
  if (r2 > kNearDiagonals * kNearDiagonals * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2])) {
    const double r = std::sqrt(r2), q = V / (4.0 * kPi * r2 * r);
    for (int a = 0; a < 3; ++a) N[a] = q * (1.0 - 3.0 * R[a] * R[a] / r2);
    N[3] = -3.0 * q * R[0] * R[1] / r2; N[4] = -3.0 * q * R[0] * R[2] / r2; N[5] = -3.0 * q * R[1] * R[2] / r2;
    return;
  }
  static const int perm_diag[3][3] = {{0, 1, 2}, {1, 0, 2}, {2, 1, 0}};      // argument order of f for xx, yy, zz
  static const int perm_off[3][3] = {{0, 1, 2}, {0, 2, 1}, {1, 2, 0}};       // argument order of g for xy, xz, yz
  for (int comp = 0; comp < 6; ++comp) {
    const int* pm = comp < 3 ? perm_diag[comp] : perm_off[comp - 3];
    double acc = 0.0;
    for (int t = 0; t < 27; ++t) {
      const int u[3] = {t % 3 - 1, (t / 3) % 3 - 1, t / 9 - 1};
      double wgt = 1.0, arg[3];
      for (int a = 0; a < 3; ++a) { wgt *= (u[a] == 0 ? -2.0 : 1.0); arg[a] = R[pm[a]] + u[a] * d[pm[a]]; }
      acc += wgt * (comp < 3 ? aux_diag(arg[0], arg[1], arg[2]) : aux_offdiag(arg[0], arg[1], arg[2]));
    }
    N[comp] = -acc / (4.0 * kPi * V);
  }
}

int nice_size(int n) {                       // smallest m >= n with only the factors 2, 3, 5, 7
  for (int m = n;; ++m) {
    int q = m;
    for (int f : {2, 3, 5, 7}) while (q % f == 0) q /= f;
    if (q == 1) return m;
  }
}

// Eq. (6).  One CTA per (cell-x a, cell-z c) slab of macrocells.  Threads form a (row-lane, column-group) grid: thread
// (rl, g) sums its VEC columns over every lanes-th of the slab's mx * mz rows (a row read is one coalesced sweep of ny
// floats per component; the unrolled row loop keeps several rows in flight); the partial column sums meet in shared
// memory, where thread b adds the row lanes and the my columns of macrocell (a, b, c) in a fixed order.  Deterministic.
constexpr int kMaxRowLanes = 8;
template <int VEC>
__global__ void coarse_grain_cells(const float* __restrict__ X, uint32_t as, int nx, int ny, int nz, int nyp, int lead,
                                   int mx, int my, int mz, long long x0, int dcy, int dcz, int py, int pz,
                                   size_t comp_stride, float mu_over_V, int lanes, float* __restrict__ M) {
  extern __shared__ float col[];                                 // [lanes][3][ny]
  const int a = blockIdx.x / dcz, c = blockIdx.x - a * dcz;
  const int i0 = (int)((x0 / mx + a) * (long long)mx - x0);      // first window plane of the cell (may be < 0)
  const int rows = mx * mz, groups = ny / VEC;
  const int rl = threadIdx.x / groups, g = threadIdx.x - rl * groups;
  if (rl < lanes) {
    float s[3][VEC];
#pragma unroll
    for (int comp = 0; comp < 3; ++comp)
#pragma unroll
      for (int v = 0; v < VEC; ++v) s[comp][v] = 0.0f;
#pragma unroll 4
    for (int r = rl; r < rows; r += lanes) {
      const int i = i0 + r / mz, k = c * mz + r % mz;
      if (i >= 0 && i < nx && k < nz) {
        const size_t e = (size_t)lead + ((size_t)i * nz + k) * nyp + (size_t)g * VEC;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
          if (VEC == 4) {
            const float4 t = __ldg(reinterpret_cast<const float4*>(X + (size_t)comp * as + e));
            s[comp][0] += t.x; s[comp][1 % VEC] += t.y; s[comp][2 % VEC] += t.z; s[comp][3 % VEC] += t.w;
          } else {
            s[comp][0] += __ldg(X + (size_t)comp * as + e);
          }
        }
      }
    }
#pragma unroll
    for (int comp = 0; comp < 3; ++comp)
#pragma unroll
      for (int v = 0; v < VEC; ++v) col[((size_t)rl * 3 + comp) * ny + g * VEC + v] = s[comp][v];
  }
  __syncthreads();
  for (int b = threadIdx.x; b < dcy; b += blockDim.x) {
    float t[3] = {0.0f, 0.0f, 0.0f};
    const int j1 = min((b + 1) * my, ny);
    for (int j = b * my; j < j1; ++j)
      for (int l = 0; l < lanes; ++l)
        for (int comp = 0; comp < 3; ++comp) t[comp] += col[((size_t)l * 3 + comp) * ny + j];
    const size_t q = ((size_t)a * py + b) * pz + c;
    M[q] = t[0] * mu_over_V; M[comp_stride + q] = t[1] * mu_over_V; M[2 * comp_stride + q] = t[2] * mu_over_V;
  }
}

// Bh_a = sum_b Kh_ab Mh_b  (Kh already carries -mu_0 and the 1/(px py pz) of the unnormalised inverse transform)
__global__ void multiply_tensor(const cufftComplex* __restrict__ Kh, const cufftComplex* __restrict__ Mh,
                                cufftComplex* __restrict__ Bh, size_t n) {
  const size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (t >= n) return;
  const cufftComplex m0 = Mh[t], m1 = Mh[n + t], m2 = Mh[2 * n + t];
  const cufftComplex kxx = Kh[t], kyy = Kh[n + t], kzz = Kh[2 * n + t], kxy = Kh[3 * n + t], kxz = Kh[4 * n + t],
                     kyz = Kh[5 * n + t];
  auto mac = [](cufftComplex a, cufftComplex b, cufftComplex acc) {
    acc.x += a.x * b.x - a.y * b.y; acc.y += a.x * b.y + a.y * b.x; return acc;
  };
  const cufftComplex z = make_cuFloatComplex(0.0f, 0.0f);
  Bh[t] = mac(kxz, m2, mac(kxy, m1, mac(kxx, m0, z)));
  Bh[n + t] = mac(kyz, m2, mac(kyy, m1, mac(kxy, m0, z)));
  Bh[2 * n + t] = mac(kzz, m2, mac(kyz, m1, mac(kxz, m0, z)));
}

void plan_dims(const Ctx& c, DemagPlan& pl) {
  pl.dcx = (c.d.nx + c.d.macro[0] - 2) / c.d.macro[0] + 1;
  pl.dcy = (c.d.ny + c.d.macro[1] - 1) / c.d.macro[1];
  pl.dcz = (c.d.nz + c.d.macro[2] - 1) / c.d.macro[2];
  pl.px = nice_size(2 * pl.dcx - 1); pl.py = nice_size(2 * pl.dcy - 1); pl.pz = nice_size(2 * pl.dcz - 1);
  if (pl.pz & 1) pl.pz = nice_size(pl.pz + 1);                 // even last dimension: aligned rows for R2C / C2R
  pl.pzc = pl.pz / 2 + 1;
}

struct Carve {
  size_t M, Mh, Kh, B, work, total;
};
bool make_plans(DemagPlan& pl, size_t work[2]) {
  int n[3] = {pl.px, pl.py, pl.pz};
  if (cufftCreate(&pl.fwd) != CUFFT_SUCCESS || cufftCreate(&pl.inv) != CUFFT_SUCCESS) return false;
  cufftSetAutoAllocation(pl.fwd, 0); cufftSetAutoAllocation(pl.inv, 0);
  if (cufftMakePlanMany(pl.fwd, 3, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_R2C, 3, &work[0]) != CUFFT_SUCCESS) return false;
  if (cufftMakePlanMany(pl.inv, 3, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2R, 3, &work[1]) != CUFFT_SUCCESS) return false;
  pl.plans = true;
  return true;
}
void carve(const DemagPlan& pl, const size_t work[2], Carve& cv) {
  const size_t real = (size_t)pl.px * pl.py * pl.pz, cplx = (size_t)pl.px * pl.py * pl.pzc;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes, 256); return o; };
  cv.M = take(3 * real * sizeof(float));
  cv.Mh = take(3 * cplx * sizeof(cufftComplex));
  cv.Kh = take(6 * cplx * sizeof(cufftComplex));
  cv.B = take(3 * real * sizeof(float));
  cv.work = take(work[0] > work[1] ? work[0] : work[1]);
  cv.total = off;
}

}  // namespace

void demag_free(Ctx& c) {
  if (!c.demag) return;
  if (c.demag->plans) { cufftDestroy(c.demag->fwd); cufftDestroy(c.demag->inv); }
  delete c.demag;
  c.demag = nullptr;
}

size_t demag_workspace_bytes(Ctx& c) {
  DemagPlan pl;
  plan_dims(c, pl);
  size_t work[2] = {0, 0};
  const bool ok = make_plans(pl, work);
  if (pl.fwd) cufftDestroy(pl.fwd);
  if (pl.inv) cufftDestroy(pl.inv);
  if (!ok) return 0;
  Carve cv;
  carve(pl, work, cv);
  return cv.total;
}

asd_status demag_enable(Ctx& c, const double spacing[3], void* ws, size_t bytes) {
  if ((c.d.ny % 4 == 0 ? c.d.ny / 4 : c.d.ny) > 1024 || (size_t)c.d.ny * 12 * kMaxRowLanes > 48 * 1024) { std::snprintf(c.err, sizeof(c.err), "asd_enable_demag: ny too large for the coarse-graining kernel"); return ASD_EUNSUPPORTED; }
  demag_free(c);
  DemagPlan* pl = new DemagPlan();
  plan_dims(c, *pl);
  size_t work[2] = {0, 0};
  if (!make_plans(*pl, work)) { c.demag = pl; demag_free(c); std::snprintf(c.err, sizeof(c.err), "cuFFT plan creation failed"); return ASD_ECUDA; }
  Carve cv;
  carve(*pl, work, cv);
  c.demag = pl;
  if (bytes < cv.total) { demag_free(c); std::snprintf(c.err, sizeof(c.err), "demag workspace too small"); return ASD_ENOMEM; }
  char* base = (char*)ws;
  pl->M = (float*)(base + cv.M); pl->Mh = (cufftComplex*)(base + cv.Mh); pl->Kh = (cufftComplex*)(base + cv.Kh);
  pl->B = (float*)(base + cv.B);
  cufftSetWorkArea(pl->fwd, base + cv.work); cufftSetWorkArea(pl->inv, base + cv.work);
  for (int a = 0; a < 3; ++a) pl->cell[a] = c.d.macro[a] * spacing[a];
  pl->mu_over_V = (float)(c.d.mu_s / (pl->cell[0] * pl->cell[1] * pl->cell[2]));

  // the six tensor components on the padded, wrapped grid (fp64 on the host), scaled by -mu_0 / (px py pz)
  const size_t real = (size_t)pl->px * pl->py * pl->pz, cplx = (size_t)pl->px * pl->py * pl->pzc;
  const double scale = -4.0e-7 * kPi / (double)real;
  std::vector<float> K(6 * real, 0.0f);
  for (int a = -(pl->dcx - 1); a <= pl->dcx - 1; ++a)
    for (int b = -(pl->dcy - 1); b <= pl->dcy - 1; ++b)
      for (int g = -(pl->dcz - 1); g <= pl->dcz - 1; ++g) {
        const double R[3] = {a * pl->cell[0], b * pl->cell[1], g * pl->cell[2]};
        double N[6];
        cuboid_tensor(pl->cell, R, N);
        const size_t q = ((size_t)((a + pl->px) % pl->px) * pl->py + (size_t)((b + pl->py) % pl->py)) * pl->pz +
                         (size_t)((g + pl->pz) % pl->pz);
        for (int comp = 0; comp < 6; ++comp) K[comp * real + q] = (float)(N[comp] * scale);
      }
  // transform them once: stage the real kernels in M / B (3 at a time), R2C into Kh
  ASD_CUDA_TRY(c, cudaMemsetAsync(pl->M, 0, 3 * real * sizeof(float), c.stream));
  cufftSetStream(pl->fwd, c.stream);
  for (int half = 0; half < 2; ++half) {
    ASD_CUDA_TRY(c, cudaMemcpyAsync(pl->B, K.data() + (size_t)half * 3 * real, 3 * real * sizeof(float),
                                    cudaMemcpyHostToDevice, c.stream));
    if (cufftExecR2C(pl->fwd, pl->B, pl->Kh + (size_t)half * 3 * cplx) != CUFFT_SUCCESS) return fail_cuda(c, cudaErrorUnknown, "cufftExecR2C (tensor)");
    ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));        // K is host memory about to go out of scope
  }
  ASD_CUDA_TRY(c, cudaMemsetAsync(pl->B, 0, 3 * real * sizeof(float), c.stream));
  graphs_invalidate(c);
  return ASD_OK;
}

// Demagnetising field of the configuration in array block aX (S or S~) into demag->B, on c.launch_stream.
asd_status launch_demag(Ctx& c, int aX) {
  DemagPlan& pl = *c.demag;
  const size_t real = (size_t)pl.px * pl.py * pl.pz, cplx = (size_t)pl.px * pl.py * pl.pzc;
  {
    const int vec = (c.d.ny % 4 == 0) ? 4 : 1, groups = c.d.ny / vec;
    int lanes = 1024 / groups;
    if (lanes > kMaxRowLanes) lanes = kMaxRowLanes;
    if (lanes < 1) lanes = 1;                                   // groups <= 1024 is checked at enable time
    const int threads = (int)align_up((size_t)(groups * lanes), 32);
    const size_t smem = (size_t)lanes * 3 * c.d.ny * sizeof(float);
    const unsigned blocks = (unsigned)(pl.dcx * pl.dcz);
    if (vec == 4)
      coarse_grain_cells<4><<<blocks, threads, smem, c.launch_stream>>>(
          c.arr(aX), (uint32_t)c.as, c.d.nx, c.d.ny, c.d.nz, c.nyp, c.lead, c.d.macro[0], c.d.macro[1], c.d.macro[2],
          (long long)c.x0, pl.dcy, pl.dcz, pl.py, pl.pz, real, pl.mu_over_V, lanes, pl.M);
    else
      coarse_grain_cells<1><<<blocks, threads, smem, c.launch_stream>>>(
          c.arr(aX), (uint32_t)c.as, c.d.nx, c.d.ny, c.d.nz, c.nyp, c.lead, c.d.macro[0], c.d.macro[1], c.d.macro[2],
          (long long)c.x0, pl.dcy, pl.dcz, pl.py, pl.pz, real, pl.mu_over_V, lanes, pl.M);
  }
  ASD_LAUNCH_CHECK(c, "coarse_grain_cells");
  cufftSetStream(pl.fwd, c.launch_stream); cufftSetStream(pl.inv, c.launch_stream);
  if (cufftExecR2C(pl.fwd, pl.M, pl.Mh) != CUFFT_SUCCESS) return fail_cuda(c, cudaErrorUnknown, "cufftExecR2C");
  multiply_tensor<<<(unsigned)((cplx + 255) / 256), 256, 0, c.launch_stream>>>(pl.Kh, pl.Mh, pl.Mh, cplx);
  ASD_LAUNCH_CHECK(c, "multiply_tensor");
  if (cufftExecC2R(pl.inv, pl.Mh, pl.B) != CUFFT_SUCCESS) return fail_cuda(c, cudaErrorUnknown, "cufftExecC2R");
  return ASD_OK;
}

void demag_fill_params(const Ctx& c, StageParams& p) {
  p.dm.B = nullptr;
  if (!c.demag) return;
  const DemagPlan& pl = *c.demag;
  p.dm.B = pl.B;
  p.dm.comp_stride = (uint32_t)((size_t)pl.px * pl.py * pl.pz);
  p.dm.sx = (uint32_t)(pl.py * pl.pz); p.dm.sy = (uint32_t)pl.pz;
  magic_u31((uint32_t)c.d.macro[0], p.dm.mx_m, p.dm.mx_s);
  magic_u31((uint32_t)c.d.macro[1], p.dm.my_m, p.dm.my_s);
  magic_u31((uint32_t)c.d.macro[2], p.dm.mz_m, p.dm.mz_s);
  p.dm.x0 = (uint32_t)c.x0; p.dm.c0 = (uint32_t)(c.x0 / c.d.macro[0]);
}

// Host copy of the cell field of the CURRENT spins (tests, diagnostics); synchronises.
asd_status demag_field_host(Ctx& c, float* out, int64_t dims[3]) {
  DemagPlan& pl = *c.demag;
  dims[0] = pl.dcx; dims[1] = pl.dcy; dims[2] = pl.dcz;
  if (!out) return ASD_OK;
  c.launch_stream = c.stream;
  const asd_status st = launch_demag(c, c.aS);
  if (st != ASD_OK) return st;
  const size_t real = (size_t)pl.px * pl.py * pl.pz;
  std::vector<float> h(3 * real);
  ASD_CUDA_TRY(c, cudaMemcpyAsync(h.data(), pl.B, 3 * real * sizeof(float), cudaMemcpyDeviceToHost, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  // cells of the spare x-slot that do not overlap the window at this alignment hold no site: reported as 0
  const int ncx = (int)((c.x0 + c.d.nx - 1) / c.d.macro[0] - c.x0 / c.d.macro[0]) + 1;
  for (int a = 0; a < pl.dcx; ++a)
    for (int b = 0; b < pl.dcy; ++b)
      for (int g = 0; g < pl.dcz; ++g)
        for (int comp = 0; comp < 3; ++comp)
          out[(((size_t)a * pl.dcy + b) * pl.dcz + g) * 3 + comp] =
              a < ncx ? h[comp * real + ((size_t)a * pl.py + b) * pl.pz + g] : 0.0f;
  return ASD_OK;
}

}  // namespace asd
