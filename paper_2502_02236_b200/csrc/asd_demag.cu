// asd_demag.cu -- demagnetising field of the atomistic window (Eq. (6)-(7)).
//
//   M_c = (mu_s / V) sum_{j in c} X_j                  Eq. (6): spins -> macrocell magnetisation (V = full cell volume)
//   B_c = -mu_0 sum_c' N(r_c' - r_c) M_c'               Eq. (7): convolution with the cuboid demagnetising tensor
//
// evaluated for the configuration of EVERY Heun stage (the paper recomputes it "at every iteration") over the
// track macrocells that overlap the window (open boundaries; the frozen track's stray field is not included -- callers
// add it through the per-site B arrays).  Each site then sees the field of its macrocell.
//
// The convolution is ours from end to end (no FFT library).  A film is a few macrocells thick, a few tens wide and a few
// hundred long, so the three axes are treated differently:
//   z (thickness, dcz cells):   summed DIRECTLY -- every pair of layers (c, c') has its own 2-D kernel K_ab(., ., c - c');
//   y (width, dcy cells):       a plain DFT of length PY = 2^n >= 2 dcy - 1 (dcy real inputs -> PY/2 + 1 complex outputs:
//                               a 32 x 33 matrix-vector product per row -- cheaper than an FFT's passes at this size);
//   x (length, dcx cells):      a shared-memory radix-2 FFT of length PX = 2^n >= 2 dcx - 1.
// Per evaluation, in stream order (3 launches):
//   coarse_grain_ydft   Eq. (6) (coalesced row sweeps, fixed summation order, deterministic) and, in the same CTA, the
//                       y-DFT of the row of cells it has just formed                  -> Y[ky][field][x-cell]
//   demag_xconv         one CTA per (ky, output component): forward FFT along x of the 3 dcz input fields (decimation
//                       in frequency, in place, output left in bit-reversed order), B^_a(c) = sum_b sum_c' K^_ab(c - c')
//                       M^_b(c') with the transformed tensor stored in the SAME bit-reversed order (so no reordering
//                       pass exists anywhere), inverse FFT (decimation in time: bit-reversed in, natural out)
//                                                                                     -> Z[ky][field][x-cell]
//   demag_yinv          inverse y-DFT (complex half-spectrum -> dcy real values)      -> B[comp][x-cell][y-cell][z-cell]
// and the stage kernel adds B[cell(site)] to its exchange field.
// The tensor is computed on the host in fp64 at enable time (Newell's closed form, point dipoles in the far field --
// DESIGN.md reading D2) and transformed there with a small fp64 FFT.  N_xx, N_yy, N_zz, N_xy are even or odd in BOTH x
// and y, so their (x, y) transforms are real; N_xz and N_yz are odd in exactly one of them: purely imaginary.  One float
// per entry is stored either way.
#include <algorithm>
#include <cmath>
#include <complex>
#include <vector>

#include <cstdlib>

#include "asd_internal.cuh"

namespace asd {

struct DemagPlan {
  int dcx = 0, dcy = 0, dcz = 0;      // macrocells that can overlap the window (x: worst alignment of x0)
  int PX = 0, PY = 0, logPX = 0;      // transform lengths (powers of two), log2 PX
  int NKY = 0, F = 0, NDZ = 0;        // PY/2 + 1 retained y-frequencies, 3 dcz fields, 2 dcz - 1 layer offsets
  double cell[3] = {0, 0, 0};
  float mu_over_V = 0.0f;
  float2* Y = nullptr;                // [NKY][F][dcx]      y-transformed cell magnetisation
  float2* Z = nullptr;                // [NKY][F][dcx]      y-transformed cell field
  float* Kh = nullptr;                // [6][NDZ][NKY][PX]  transformed tensor (x index bit-reversed), includes -mu_0/(PX PY)
  float* B = nullptr;                 // [3][dcx][dcy][dcz] cell field, Tesla
  float2* twx = nullptr;              // [PX/2] exp(-2 pi i n / PX)
  float2* twy = nullptr;              // [PY]   exp(+2 pi i n / PY)
  unsigned xconv_threads = 0;
  size_t xconv_smem = 0;
  // Eq. (6) folded into the fused step (asd_heun_fused.cu): macrocell sums of the spins the last fused step wrote
  long long* acc = nullptr;           // [3][dcx][dcy][dcz], units of 1 / acc_fx
  float acc_fx = 0.0f;                // a power of two; a whole cell's sum stays below 2^31
  enum AccState { ACC_CLEAN, ACC_VALID, ACC_STALE } acc_state = ACC_CLEAN;   // zeros / sums of the current S / leftovers
  // stray field of the frozen track on the window's macrocells (reading D4); own workspace
  bool stray = false;
  int XR = 0;                         // largest |x offset| in cells between a source and a target cell
  float* Nt = nullptr;                // [2 XR + 1][2 dcy - 1][2 dcz - 1][6] cuboid tensor times -mu_0 mu_s / V
  float* mom = nullptr;               // [track cells][3] sum of the frozen spins of a cell that lie outside the window
  float* Bt = nullptr;                // [3][dcx][dcy][dcz] the track's stray field, Tesla (added by demag_yinv)
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


int pow2_at_least(int n) { int p = 2; while (p < n) p <<= 1; return p; }

// in-place iterative radix-2 FFT, fp64, forward (e^{-i...}); host, set-up only
void host_fft(std::complex<double>* x, int n) {
  for (int i = 1, j = 0; i < n; ++i) {
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) std::swap(x[i], x[j]);
  }
  for (int len = 2; len <= n; len <<= 1) {
    const double ang = -2.0 * kPi / len;
    for (int i = 0; i < n; i += len)
      for (int k = 0; k < len / 2; ++k) {
        const std::complex<double> w(std::cos(ang * k), std::sin(ang * k));
        const std::complex<double> u = x[i + k], v = x[i + k + len / 2] * w;
        x[i + k] = u + v; x[i + k + len / 2] = u - v;
      }
  }
}

uint32_t bit_reverse(uint32_t v, int bits) {
  uint32_t r = 0;
  for (int b = 0; b < bits; ++b) r |= ((v >> b) & 1u) << (bits - 1 - b);
  return r;
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cmul_conj(float2 a, float2 w) { return make_float2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// y-DFT of one row of dcy cell values per component (shared memory `cells` [3][dcy]) into Y[ky][comp dcz + c][a]:
//   Y = sum_b M_comp(a, b, c) exp(-2 pi i ky b / PY),  ky = 0 .. PY/2.
// Four threads share an output (every fourth b each, combined by shuffles in a fixed order); tws = exp(+i ...) table in
// shared memory.  Called by all threads of the CTA (blockDim a multiple of 32).
__device__ __forceinline__ void row_ydft(const float* cells, const float2* tws, int dcy, int dcz, int dcx, int PY, int NKY,
                                         int a, int c, float2* __restrict__ Y) {
  const int F = 3 * dcz, nout = 3 * NKY;
  for (int o4 = threadIdx.x; o4 < ((4 * nout + 31) & ~31); o4 += blockDim.x) {
    const int o = o4 >> 2, part = o4 & 3;
    const int comp = o < nout ? o / NKY : 0, ky = o < nout ? o - comp * NKY : 0;
    float re = 0.0f, im = 0.0f;
    for (int b = part; b < dcy; b += 4) {
      const float2 w = tws[(ky * b) & (PY - 1)];
      const float m = cells[comp * dcy + b];
      re = fmaf(m, w.x, re); im = fmaf(-m, w.y, im);
    }
    re += __shfl_xor_sync(0xFFFFFFFFu, re, 1); im += __shfl_xor_sync(0xFFFFFFFFu, im, 1);
    re += __shfl_xor_sync(0xFFFFFFFFu, re, 2); im += __shfl_xor_sync(0xFFFFFFFFu, im, 2);
    if (part == 0 && o < nout) Y[((size_t)ky * F + (size_t)(comp * dcz + c)) * dcx + a] = make_float2(re, im);
  }
}

// Eq. (6) + the y-DFT.  One CTA per (cell-x a, cell-z c) slab of macrocells.  Threads form a (row-lane, column-group)
// grid: thread (rl, g) sums its VEC columns over every lanes-th of the slab's mx * mz rows (a row read is one coalesced
// sweep of ny floats per component; the unrolled row loop keeps several rows in flight); the partial column sums meet in
// shared memory, where thread b adds the row lanes and the my columns of macrocell (a, b, c) in a fixed order.
// Deterministic.  The dcy cell values of each component are then transformed along y (row_ydft).
constexpr int kMaxRowLanes = 4;   // measured on cfg4 (B200): 3-4 lanes 141.6-142.0 us per held-field Heun step, 8 lanes 146.3, 1 lane 155.6
template <int VEC>
__global__ void coarse_grain_ydft(const float* __restrict__ X, uint32_t as, int nx, int ny, int nz, int nyp, int lead,
                                  int mx, int my, int mz, long long x0, int dcx, int dcy, int dcz, int PY, int NKY,
                                  float mu_over_V, int lanes, const float2* __restrict__ twy, float2* __restrict__ Y) {
  extern __shared__ __align__(16) float col[];                   // [lanes][3][ny] | cells [3][dcy] | tws [PY]
  float* cells = col + (size_t)lanes * 3 * ny;
  float2* tws = reinterpret_cast<float2*>(cells + ((3 * dcy + 1) & ~1));
  const int a = blockIdx.x / dcz, c = blockIdx.x - a * dcz;
  const int i0 = (int)((x0 / mx + a) * (long long)mx - x0);      // first window plane of the cell (may be < 0)
  const int rows = mx * mz, groups = ny / VEC;
  const int rl = threadIdx.x / groups, g = threadIdx.x - rl * groups;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  for (int t = threadIdx.x; t < PY; t += blockDim.x) tws[t] = __ldg(twy + t);
  asm volatile("griddepcontrol.wait;" ::: "memory");            // the kernel that wrote X has completed
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
  for (int t = threadIdx.x; t < 3 * dcy; t += blockDim.x) {      // one thread per (component, macrocell): fixed order
    const int comp = t / dcy, b = t - comp * dcy;
    float acc = 0.0f;
    const int j1 = min((b + 1) * my, ny);
    for (int j = b * my; j < j1; ++j)
      for (int l = 0; l < lanes; ++l) acc += col[((size_t)l * 3 + comp) * ny + j];
    cells[t] = acc * mu_over_V;
  }
  __syncthreads();
  row_ydft(cells, tws, dcy, dcz, dcx, PY, NKY, a, c, Y);
}

// The same from the cell sums the fused step's corrector accumulated (64-bit fixed point, 1 / fx units): one CTA per
// (cell-x a, cell-z c).  The sums are cleared for the next accumulation by demag_xconv, which follows: scattered 8-byte
// stores from here kept every CTA waiting at its exit (measured: 10.1 us with them, 6.3 without).
__global__ void cells_ydft(const long long* __restrict__ acc, double scale, int dcx, int dcy, int dcz, int PY, int NKY,
                           const float2* __restrict__ twy, float2* __restrict__ Y) {
  extern __shared__ __align__(16) float col[];                   // cells [3][dcy] | tws [PY]
  float* cells = col;
  float2* tws = reinterpret_cast<float2*>(cells + ((3 * dcy + 1) & ~1));
  const int a = blockIdx.x / dcz, c = blockIdx.x - a * dcz;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  for (int t = threadIdx.x; t < PY; t += blockDim.x) tws[t] = __ldg(twy + t);
  asm volatile("griddepcontrol.wait;" ::: "memory");            // the step that accumulated the sums has completed
  for (int t = threadIdx.x; t < 3 * dcy; t += blockDim.x) {
    const int comp = t / dcy, b = t - comp * dcy;
    const size_t q = (((size_t)comp * dcx + a) * dcy + b) * dcz + c;
    cells[t] = (float)((double)acc[q] * scale);
  }
  __syncthreads();
  row_ydft(cells, tws, dcy, dcz, dcx, PY, NKY, a, c, Y);
}

// Which stored tensor component couples output component oc to input component b.  Storage order
// (Nxx, Nyy, Nzz, Nxy, Nxz, Nyz); the (x, y) transforms of the last two are purely imaginary.
__device__ __forceinline__ int tensor_comp(int oc, int b) {
  return oc == b ? oc : (oc + b == 1 ? 3 : (oc + b == 2 ? 4 : 5));
}

// ---- shared-memory FFT along x ----
// A field of PX complex points is stored with one pad element after every 8 (phys): the 8-point chunks that one thread
// transforms in registers then start 72 bytes apart, which makes their 64-bit accesses bank-conflict-free, and the
// wide-span stages (consecutive threads, consecutive points) lose next to nothing.
__device__ __forceinline__ int phys(int n) { return n + (n >> 3); }

// Decimation in frequency (forward, e^{-i}): stage of span h maps the pair (p, p + h), p mod 2h < h, to
// (a + b, (a - b) w),  w = exp(-2 pi i (p mod h) / (2 h)) = tw[(p mod h) (PX / 2h)];  natural order in, bit-reversed out.
// Decimation in time (inverse, e^{+i}): the same pairs, (a + b conj w, a - b conj w), spans ascending.
__device__ __forceinline__ void dif_stage(float2* x, int f_count, int logPX, int sh, const float2* tw, int PXP) {
  const int H = 1 << (logPX - 1), h = 1 << sh;
  for (int t = threadIdx.x; t < f_count * H; t += blockDim.x) {
    const int f = t >> (logPX - 1), u = t & (H - 1);
    const int i = u & (h - 1), p = ((u >> sh) << (sh + 1)) + i;
    float2* xf = x + f * PXP;
    const float2 a = xf[phys(p)], b = xf[phys(p + h)];
    xf[phys(p)] = cadd(a, b);
    xf[phys(p + h)] = cmul(csub(a, b), tw[i << (logPX - 1 - sh)]);
  }
}
__device__ __forceinline__ void dit_stage(float2* x, int f_count, int logPX, int sh, const float2* tw, int PXP) {
  const int H = 1 << (logPX - 1), h = 1 << sh;
  for (int t = threadIdx.x; t < f_count * H; t += blockDim.x) {
    const int f = t >> (logPX - 1), u = t & (H - 1);
    const int i = u & (h - 1), p = ((u >> sh) << (sh + 1)) + i;
    float2* xf = x + f * PXP;
    const float2 a = xf[phys(p)], b = cmul_conj(xf[phys(p + h)], tw[i << (logPX - 1 - sh)]);
    xf[phys(p)] = cadd(a, b);
    xf[phys(p + h)] = csub(a, b);
  }
}
// Two stages at once (spans h = 2^sh and h/2), four points per work item in registers.
__device__ __forceinline__ void dif_pair(float2* x, int f_count, int logPX, int sh, const float2* tw, int PXP) {
  const int Q = 1 << (logPX - 2), h = 1 << sh, hh = h >> 1;
  for (int t = threadIdx.x; t < f_count * Q; t += blockDim.x) {
    const int f = t >> (logPX - 2), u = t & (Q - 1);
    const int i = u & (hh - 1), p0 = ((u >> (sh - 1)) << (sh + 1)) + i;
    float2* xf = x + f * PXP;
    const int q0 = phys(p0), q1 = phys(p0 + hh), q2 = phys(p0 + h), q3 = phys(p0 + h + hh);
    const float2 x0 = xf[q0], x1 = xf[q1], x2 = xf[q2], x3 = xf[q3];
    const int ts = logPX - 1 - sh;                                // twiddle stride of span h
    const float2 a0 = cadd(x0, x2), a2 = cmul(csub(x0, x2), tw[i << ts]);
    const float2 a1 = cadd(x1, x3), a3 = cmul(csub(x1, x3), tw[(i + hh) << ts]);
    const float2 w = tw[i << (ts + 1)];
    xf[q0] = cadd(a0, a1); xf[q1] = cmul(csub(a0, a1), w);
    xf[q2] = cadd(a2, a3); xf[q3] = cmul(csub(a2, a3), w);
  }
}
// spans h = 2^sh and 2h
__device__ __forceinline__ void dit_pair(float2* x, int f_count, int logPX, int sh, const float2* tw, int PXP) {
  const int Q = 1 << (logPX - 2), h = 1 << sh;
  for (int t = threadIdx.x; t < f_count * Q; t += blockDim.x) {
    const int f = t >> (logPX - 2), u = t & (Q - 1);
    const int i = u & (h - 1), p0 = ((u >> sh) << (sh + 2)) + i;
    float2* xf = x + f * PXP;
    const int q0 = phys(p0), q1 = phys(p0 + h), q2 = phys(p0 + 2 * h), q3 = phys(p0 + 3 * h);
    const float2 x0 = xf[q0], x1 = xf[q1], x2 = xf[q2], x3 = xf[q3];
    const int ts = logPX - 1 - sh;
    const float2 w = tw[i << ts];
    const float2 b1 = cmul_conj(x1, w), b3 = cmul_conj(x3, w);
    const float2 a0 = cadd(x0, b1), a1 = csub(x0, b1), a2 = cadd(x2, b3), a3 = csub(x2, b3);
    const float2 c2 = cmul_conj(a2, tw[i << (ts - 1)]), c3 = cmul_conj(a3, tw[(i + h) << (ts - 1)]);
    xf[q0] = cadd(a0, c2); xf[q2] = csub(a0, c2);
    xf[q1] = cadd(a1, c3); xf[q3] = csub(a1, c3);
  }
}
// Spans 4, 2, 1 (forward) / 1, 2, 4 (inverse) of one aligned 8-point chunk, in registers.
constexpr float kR = 0.70710678118654752440f;
template <bool INV>
__device__ __forceinline__ void chunk8(float2* x, int f_count, int logPX, int PXP) {
  const int C = 1 << (logPX - 3);
  for (int t = threadIdx.x; t < f_count * C; t += blockDim.x) {
    const int f = t >> (logPX - 3), u = t & (C - 1);
    float2* xc = x + f * PXP + 9 * u;                            // phys(8 u) = 9 u; the 8 points are contiguous
    float2 v[8];
#pragma unroll
    for (int n = 0; n < 8; ++n) v[n] = xc[n];
    // w8[i] = exp(-2 pi i i / 8)
    const float2 w8[4] = {make_float2(1.f, 0.f), make_float2(kR, -kR), make_float2(0.f, -1.f), make_float2(-kR, -kR)};
    if (!INV) {
#pragma unroll
      for (int i = 0; i < 4; ++i) { const float2 a = v[i], b = v[i + 4]; v[i] = cadd(a, b); v[i + 4] = cmul(csub(a, b), w8[i]); }
#pragma unroll
      for (int blk = 0; blk < 8; blk += 4)
#pragma unroll
        for (int i = 0; i < 2; ++i) { const float2 a = v[blk + i], b = v[blk + i + 2]; v[blk + i] = cadd(a, b); v[blk + i + 2] = cmul(csub(a, b), w8[2 * i]); }
#pragma unroll
      for (int blk = 0; blk < 8; blk += 2) { const float2 a = v[blk], b = v[blk + 1]; v[blk] = cadd(a, b); v[blk + 1] = csub(a, b); }
    } else {
#pragma unroll
      for (int blk = 0; blk < 8; blk += 2) { const float2 a = v[blk], b = v[blk + 1]; v[blk] = cadd(a, b); v[blk + 1] = csub(a, b); }
#pragma unroll
      for (int blk = 0; blk < 8; blk += 4)
#pragma unroll
        for (int i = 0; i < 2; ++i) { const float2 a = v[blk + i], b = cmul_conj(v[blk + i + 2], w8[2 * i]); v[blk + i] = cadd(a, b); v[blk + i + 2] = csub(a, b); }
#pragma unroll
      for (int i = 0; i < 4; ++i) { const float2 a = v[i], b = cmul_conj(v[i + 4], w8[i]); v[i] = cadd(a, b); v[i + 4] = csub(a, b); }
    }
#pragma unroll
    for (int n = 0; n < 8; ++n) xc[n] = v[n];
  }
}

// One CTA per (ky, output component oc): x-FFT of all F = 3 dcz input fields, the tensor product with the direct sum
// over layers, inverse x-FFT of the dcz output fields of component oc.
__global__ void __launch_bounds__(1024, 1)
demag_xconv(const float2* __restrict__ Y, float2* __restrict__ Z, const float* __restrict__ Kh,
            const float2* __restrict__ twx, int dcx, int dcz, int PX, int logPX, int NKY,
            long long* __restrict__ acc_clear, int acc_n) {
  extern __shared__ __align__(16) float2 xs[];                   // X[F][PXP] | O[dcz][PXP] | tw[PX/2] | Ks[3][NDZ][PX]
  const int F = 3 * dcz, NDZ = 2 * dcz - 1, H = PX >> 1, PXP = PX + (PX >> 3);
  float2* X = xs;
  float2* O = X + (size_t)F * PXP;
  float2* tw = O + (size_t)dcz * PXP;
  float* Ks = reinterpret_cast<float*>(tw + H);
  const int ky = blockIdx.x, oc = blockIdx.y;
  const int tid = threadIdx.x, nt = blockDim.x;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // constants of the context (not written by the previous kernel): twiddles, and this CTA's slice of the transformed
  // tensor -- 3 input components x NDZ layer offsets x PX points -- by asynchronous 16-byte copies that land while the
  // forward transform runs
  for (int t = tid; t < H; t += nt) tw[t] = __ldg(twx + t);
  for (int t = tid; t < 3 * NDZ * (PX >> 2); t += nt) {
    const int row = t / (PX >> 2), q = t - row * (PX >> 2);      // row = b NDZ + dzi
    const int b = row / NDZ, dzi = row - b * NDZ;
    const float* src = Kh + (((size_t)tensor_comp(oc, b) * NDZ + dzi) * NKY + ky) * PX + 4 * q;
    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(Ks + (size_t)row * PX + 4 * q);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (acc_clear) {
    // cells_ydft has read the fused step's cell sums: cleared here (coalesced, long before this kernel ends)
    const int gt = (blockIdx.y * gridDim.x + blockIdx.x) * nt + tid, gn = gridDim.x * gridDim.y * nt;
    for (int t = gt; t < acc_n; t += gn) acc_clear[t] = 0;
  }
  __syncthreads();
  // Load with the first forward stage folded in: the upper half of the padded input is zero (dcx <= PX/2), so that
  // stage is X[p] = x[p], X[p + PX/2] = x[p] w^p.
  for (int t = tid; t < F * H; t += nt) {
    const int f = t >> (logPX - 1), p = t & (H - 1);
    const float2 v = p < dcx ? Y[((size_t)ky * F + f) * dcx + p] : make_float2(0.0f, 0.0f);
    X[f * PXP + phys(p)] = v;
    X[f * PXP + phys(p + H)] = cmul(v, tw[p]);
  }
  __syncthreads();
  if (logPX >= 4) {
    int sh = logPX - 2;
    while (sh >= 4) { dif_pair(X, F, logPX, sh, tw, PXP); sh -= 2; __syncthreads(); }
    if (sh == 3) { dif_stage(X, F, logPX, 3, tw, PXP); __syncthreads(); }
    chunk8<false>(X, F, logPX, PXP);
  } else {
    for (int sh = logPX - 2; sh >= 0; --sh) { dif_stage(X, F, logPX, sh, tw, PXP); __syncthreads(); }
  }
  asm volatile("cp.async.wait_all;" ::: "memory");
  __syncthreads();
  // X[f][p] now holds the spectrum at kx = bitrev(p); Ks is in the same order.  One work item per (output layer c, p).
  for (int t = tid; t < dcz * PX; t += nt) {
    const int c = t >> logPX, p = t & (PX - 1), pp = phys(p);
    float2 acc = make_float2(0.0f, 0.0f);
    for (int b = 0; b < 3; ++b) {
      const bool imag = tensor_comp(oc, b) >= 4;
      const float* kp = Ks + (size_t)(b * NDZ + c + dcz - 1) * PX + p;      // dz = c - c' -> dzi = c - c' + dcz - 1
      const float2* xp = X + (size_t)(b * dcz) * PXP + pp;
      float2 s = make_float2(0.0f, 0.0f);
      for (int cp = 0; cp < dcz; ++cp) {
        const float kap = kp[-cp * PX];
        const float2 x = xp[cp * PXP];
        s.x = fmaf(kap, x.x, s.x); s.y = fmaf(kap, x.y, s.y);
      }
      if (imag) { acc.x -= s.y; acc.y += s.x; } else { acc.x += s.x; acc.y += s.y; }
    }
    O[c * PXP + pp] = acc;
  }
  __syncthreads();
  if (logPX >= 4) {
    chunk8<true>(O, dcz, logPX, PXP);
    __syncthreads();
    int sh = 3;
    while (sh + 1 <= logPX - 1) { dit_pair(O, dcz, logPX, sh, tw, PXP); sh += 2; __syncthreads(); }
    if (sh == logPX - 1) { dit_stage(O, dcz, logPX, sh, tw, PXP); __syncthreads(); }
  } else {
    for (int sh = 0; sh < logPX; ++sh) { dit_stage(O, dcz, logPX, sh, tw, PXP); __syncthreads(); }
  }
  for (int t = tid; t < dcz * dcx; t += nt) {
    const int c = t / dcx, a = t - c * dcx;
    Z[((size_t)ky * F + (size_t)(oc * dcz + c)) * dcx + a] = O[c * PXP + phys(a)];
  }
}

// Inverse y-DFT of the half spectrum: B_f(a, b) = Re sum_ky wgt_ky Z[ky][f][a] exp(+2 pi i ky b / PY), wgt = 1 for
// ky = 0 and PY/2, 2 otherwise (Hermitian symmetry of a real field).  One CTA per (field f, 8 x-cells); one output per
// thread and pass.
constexpr int kYinvCols = 8;
__global__ void demag_yinv(const float2* __restrict__ Z, const float2* __restrict__ twy, float* __restrict__ B,
                           int dcx, int dcy, int dcz, int PY, int NKY, const float* __restrict__ Bt) {
  extern __shared__ __align__(16) float2 zs[];                   // [NKY][8] | tws[PY]
  float2* tws = zs + NKY * kYinvCols;
  const int F = 3 * dcz, f = blockIdx.y, a0 = blockIdx.x * kYinvCols;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  for (int t = threadIdx.x; t < PY; t += blockDim.x) tws[t] = __ldg(twy + t);
  asm volatile("griddepcontrol.wait;" ::: "memory");
  for (int t = threadIdx.x; t < NKY * kYinvCols; t += blockDim.x) {
    const int ky = t / kYinvCols, da = t - ky * kYinvCols;
    float2 v = make_float2(0.0f, 0.0f);
    if (a0 + da < dcx) v = Z[((size_t)ky * F + f) * dcx + a0 + da];
    const float wgt = (ky == 0 || ky == NKY - 1) ? 1.0f : 2.0f;
    zs[t] = make_float2(wgt * v.x, wgt * v.y);
  }
  __syncthreads();
  const int comp = f / dcz, c = f - comp * dcz;
  for (int t = threadIdx.x; t < dcy * kYinvCols; t += blockDim.x) {
    const int b = t / kYinvCols, da = t - b * kYinvCols;
    if (a0 + da >= dcx) continue;
    float acc0 = 0.0f, acc1 = 0.0f;
    int ky = 0;
    for (; ky + 1 < NKY; ky += 2) {
      const float2 w0 = tws[(ky * b) & (PY - 1)], w1 = tws[((ky + 1) * b) & (PY - 1)];
      const float2 z0 = zs[ky * kYinvCols + da], z1 = zs[(ky + 1) * kYinvCols + da];
      acc0 = fmaf(z0.x, w0.x, fmaf(-z0.y, w0.y, acc0));
      acc1 = fmaf(z1.x, w1.x, fmaf(-z1.y, w1.y, acc1));
    }
    if (ky < NKY) {
      const float2 w0 = tws[(ky * b) & (PY - 1)];
      const float2 z0 = zs[ky * kYinvCols + da];
      acc0 = fmaf(z0.x, w0.x, fmaf(-z0.y, w0.y, acc0));
    }
    const size_t o = (((size_t)comp * dcx + (a0 + da)) * dcy + b) * dcz + c;
    B[o] = acc0 + acc1 + (Bt ? Bt[o] : 0.0f);            // + the frozen track's stray field (static between shifts)
  }
}

// ---- stray field of the frozen track (reading D4) ----
// Outside moment of every track cell in columns [cx_lo, cx_hi]: what has left the window (out_sum: the frozen spins
// themselves) plus the init mean spin times the number of magnetic sites the window has never held.
__global__ void stray_moments_kernel(const uint32_t* __restrict__ col_track, const double* __restrict__ out_sum,
                                     const long long* __restrict__ out_cnt, const float* __restrict__ init_mean,
                                     float* __restrict__ mom, long long cx_lo, long long cx_hi, int ncy, int ncz, int mx,
                                     int my, int mz, int ny, int nz, long long track_nx, long long x0, int nx) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long n = (cx_hi - cx_lo + 1) * ncy * ncz;
  if (r >= n) return;
  const int c2 = (int)(r % ncz), b2 = (int)((r / ncz) % ncy);
  const long long cx = cx_lo + r / ((long long)ncz * ncy);
  const int kext = min((c2 + 1) * mz, nz) - c2 * mz;
  long long n_out = 0;
  for (long long gx = cx * mx; gx < min((cx + 1) * (long long)mx, track_nx); ++gx) {
    if (gx >= x0 && gx < x0 + nx) continue;
    for (int j = b2 * my; j < min((b2 + 1) * my, ny); ++j)
      if ((col_track[gx * ny + j] & 0xFFFFu) != 0u) n_out += kext;
  }
  const long long t = (cx * ncy + b2) * ncz + c2;
  const double fresh = (double)(n_out - out_cnt[t]);
  for (int u = 0; u < 3; ++u) mom[3 * t + u] = (float)(out_sum[3 * t + u] + (double)init_mean[3 * t + u] * fresh);
}

// B_c = sum_c' Nt(r_c' - r_c) mom_c' for the window cells of one x column (blockIdx.x = a); thread = (b, c).  Source
// columns are taken one at a time through shared memory, in ascending order (deterministic); all-zero columns (the
// window's interior) are skipped.
__global__ void stray_sum_kernel(const float* __restrict__ Nt, const float* __restrict__ mom, float* __restrict__ Bt,
                                 long long c0, long long cx_lo, long long cx_hi, int XR, int dcx, int dcy, int dcz,
                                 int ncy, int ncz) {
  extern __shared__ float sm_mom[];                              // [ncy*ncz][3]
  const int a = blockIdx.x, ncol = ncy * ncz;
  const int sy = 2 * dcy - 1, sz = 2 * dcz - 1;
  for (int tgt0 = 0; tgt0 < dcy * dcz; tgt0 += blockDim.x) {
    const int tgt = tgt0 + threadIdx.x;
    const bool on = tgt < dcy * dcz;
    const int b = on ? tgt / dcz : 0, c = on ? tgt - b * dcz : 0;
    float acc[3] = {0.f, 0.f, 0.f};
    for (long long cx = cx_lo; cx <= cx_hi; ++cx) {
      const long long dx = cx - (c0 + a);
      if (dx > XR || dx < -XR) continue;                          // uniform over the block
      int nz_any = 0;
      __syncthreads();
      for (int t = threadIdx.x; t < 3 * ncol; t += blockDim.x) {
        const float v = mom[3 * cx * ncol + t];
        sm_mom[t] = v;
        nz_any |= (v != 0.0f);
      }
      if (!__syncthreads_or(nz_any)) continue;
      if (on) {
        const float* Nx = Nt + (size_t)(dx + XR) * sy * sz * 6;
        for (int b2 = 0; b2 < ncy; ++b2)
          for (int c2 = 0; c2 < ncz; ++c2) {
            const float* N = Nx + ((size_t)(b2 - b + dcy - 1) * sz + (c2 - c + dcz - 1)) * 6;
            const float m0 = sm_mom[3 * (b2 * ncz + c2)], m1 = sm_mom[3 * (b2 * ncz + c2) + 1], m2 = sm_mom[3 * (b2 * ncz + c2) + 2];
            acc[0] = fmaf(N[0], m0, fmaf(N[3], m1, fmaf(N[4], m2, acc[0])));
            acc[1] = fmaf(N[3], m0, fmaf(N[1], m1, fmaf(N[5], m2, acc[1])));
            acc[2] = fmaf(N[4], m0, fmaf(N[5], m1, fmaf(N[2], m2, acc[2])));
          }
      }
    }
    if (on)
      for (int u = 0; u < 3; ++u) Bt[(((size_t)u * dcx + a) * dcy + b) * dcz + c] = acc[u];
  }
}

void plan_dims(const Ctx& c, DemagPlan& pl) {
  pl.dcx = (c.d.nx + c.d.macro[0] - 2) / c.d.macro[0] + 1;
  pl.dcy = (c.d.ny + c.d.macro[1] - 1) / c.d.macro[1];
  pl.dcz = (c.d.nz + c.d.macro[2] - 1) / c.d.macro[2];
  pl.PX = std::max(4, pow2_at_least(2 * pl.dcx - 1)); pl.PY = pow2_at_least(2 * pl.dcy - 1);   // PX >= 4: 16-byte rows of the tensor slice
  pl.logPX = 0;
  while ((1 << pl.logPX) < pl.PX) ++pl.logPX;
  pl.NKY = pl.PY / 2 + 1; pl.F = 3 * pl.dcz; pl.NDZ = 2 * pl.dcz - 1;
  const size_t PXP = (size_t)pl.PX + pl.PX / 8;
  pl.xconv_smem = ((size_t)(pl.F + pl.dcz) * PXP + pl.PX / 2) * sizeof(float2) + (size_t)3 * pl.NDZ * pl.PX * sizeof(float);
  // one 8-point chunk per thread in the register stage (two 4-point items in the paired stages)
  const size_t chunks = (size_t)pl.F * std::max(pl.PX / 8, 1);
  pl.xconv_threads = (unsigned)std::min<size_t>(1024, std::max<size_t>(128, (chunks + 31) / 32 * 32));
}

size_t cg_smem_bytes(int lanes, int ny, const DemagPlan& pl) {
  return ((size_t)lanes * 3 * ny + ((3 * (size_t)pl.dcy + 1) & ~(size_t)1)) * sizeof(float) + (size_t)pl.PY * sizeof(float2);
}

struct Carve {
  size_t Y, Z, Kh, B, twx, twy, acc, total;
};
void carve(const DemagPlan& pl, Carve& cv) {
  const size_t spec = (size_t)pl.NKY * pl.F * pl.dcx;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes, 256); return o; };
  cv.Y = take(spec * sizeof(float2));
  cv.Z = take(spec * sizeof(float2));
  cv.Kh = take((size_t)6 * pl.NDZ * pl.NKY * pl.PX * sizeof(float));
  cv.B = take((size_t)3 * pl.dcx * pl.dcy * pl.dcz * sizeof(float));
  cv.twx = take((size_t)(pl.PX / 2) * sizeof(float2));
  cv.twy = take((size_t)pl.PY * sizeof(float2));
  cv.acc = take((size_t)3 * pl.dcx * pl.dcy * pl.dcz * sizeof(long long));
  cv.total = off;
}

}  // namespace

void demag_free(Ctx& c) {
  delete c.demag;
  c.demag = nullptr;
}

size_t demag_workspace_bytes(Ctx& c) {
  DemagPlan pl;
  plan_dims(c, pl);
  Carve cv;
  carve(pl, cv);
  return cv.total;
}

asd_status demag_enable(Ctx& c, const double spacing[3], void* ws, size_t bytes) {
  if ((c.d.ny % 4 == 0 ? c.d.ny / 4 : c.d.ny) > 1024) { std::snprintf(c.err, sizeof(c.err), "asd_enable_demag: ny too large for the coarse-graining kernel"); return ASD_EUNSUPPORTED; }
  demag_free(c);
  DemagPlan* pl = new DemagPlan();
  plan_dims(c, *pl);
  int smem_cta = 0;
  cudaDeviceGetAttribute(&smem_cta, cudaDevAttrMaxSharedMemoryPerBlockOptin, c.device);
  const size_t cg_smem = cg_smem_bytes(kMaxRowLanes, c.d.ny, *pl);
  if (pl->xconv_smem > (size_t)smem_cta || cg_smem > (size_t)smem_cta) {
    delete pl;
    std::snprintf(c.err, sizeof(c.err), "asd_enable_demag: window too long / thick for the shared-memory transform (3 dcz fields x PX points must fit in %d bytes)", smem_cta);
    return ASD_EUNSUPPORTED;
  }
  Carve cv;
  carve(*pl, cv);
  if (bytes < cv.total) { delete pl; std::snprintf(c.err, sizeof(c.err), "demag workspace too small"); return ASD_ENOMEM; }
  c.demag = pl;
  char* base = (char*)ws;
  pl->Y = (float2*)(base + cv.Y); pl->Z = (float2*)(base + cv.Z); pl->Kh = (float*)(base + cv.Kh);
  pl->B = (float*)(base + cv.B); pl->twx = (float2*)(base + cv.twx); pl->twy = (float2*)(base + cv.twy);
  pl->acc = (long long*)(base + cv.acc);
  {
    const long long sites = (long long)c.d.macro[0] * c.d.macro[1] * c.d.macro[2];
    int bits = 30;
    while (bits > 0 && (sites << bits) >= (1ll << 31)) --bits;
    pl->acc_fx = (float)(1ll << bits);
  }
  for (int a = 0; a < 3; ++a) pl->cell[a] = c.d.macro[a] * spacing[a];
  pl->mu_over_V = (float)(c.d.mu_s / (pl->cell[0] * pl->cell[1] * pl->cell[2]));
  ASD_CUDA_TRY(c, cudaFuncSetAttribute((const void*)demag_xconv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->xconv_smem));
  ASD_CUDA_TRY(c, cudaFuncSetAttribute((const void*)coarse_grain_ydft<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cg_smem));
  ASD_CUDA_TRY(c, cudaFuncSetAttribute((const void*)coarse_grain_ydft<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cg_smem));

  // The six tensor components for every cell offset (fp64, host), one (x, y) plane per layer offset dz: wrapped onto the
  // PX x PY grid, transformed, scaled by -mu_0 / (PX PY) (both inverse transforms are unnormalised), reduced to the real
  // or imaginary part that survives, and stored with the x index bit-reversed (the order demag_xconv's forward transform
  // leaves its spectra in).
  const int PX = pl->PX, PY = pl->PY, NKY = pl->NKY, NDZ = pl->NDZ;
  const double scale = -4.0e-7 * kPi / ((double)PX * PY);
  std::vector<float> Kh((size_t)6 * NDZ * NKY * PX, 0.0f);
  std::vector<std::complex<double>> plane((size_t)6 * PX * PY), line((size_t)std::max(PX, PY));
  std::vector<uint32_t> rev(PX);
  for (int p = 0; p < PX; ++p) rev[p] = bit_reverse((uint32_t)p, pl->logPX);
  for (int dzi = 0; dzi < NDZ; ++dzi) {
    const int g = dzi - (pl->dcz - 1);
    std::fill(plane.begin(), plane.end(), std::complex<double>(0.0, 0.0));
    for (int a = -(pl->dcx - 1); a <= pl->dcx - 1; ++a)
      for (int b = -(pl->dcy - 1); b <= pl->dcy - 1; ++b) {
        const double R[3] = {a * pl->cell[0], b * pl->cell[1], g * pl->cell[2]};
        double N[6];
        cuboid_tensor(pl->cell, R, N);
        const size_t q = (size_t)((a + PX) % PX) * PY + (size_t)((b + PY) % PY);
        for (int comp = 0; comp < 6; ++comp) plane[(size_t)comp * PX * PY + q] = N[comp] * scale;
      }
    for (int comp = 0; comp < 6; ++comp) {
      std::complex<double>* P = plane.data() + (size_t)comp * PX * PY;
      for (int x = 0; x < PX; ++x) host_fft(P + (size_t)x * PY, PY);
      for (int y = 0; y < NKY; ++y) {
        for (int x = 0; x < PX; ++x) line[x] = P[(size_t)x * PY + y];
        host_fft(line.data(), PX);
        float* dst = Kh.data() + (((size_t)comp * NDZ + dzi) * NKY + y) * PX;
        for (int p = 0; p < PX; ++p) dst[p] = (float)(comp >= 4 ? line[rev[p]].imag() : line[rev[p]].real());
      }
    }
  }
  std::vector<float2> twx(PX / 2), twy(PY);
  for (int n = 0; n < PX / 2; ++n) twx[n] = make_float2((float)std::cos(-2.0 * kPi * n / PX), (float)std::sin(-2.0 * kPi * n / PX));
  for (int n = 0; n < PY; ++n) twy[n] = make_float2((float)std::cos(2.0 * kPi * n / PY), (float)std::sin(2.0 * kPi * n / PY));
  ASD_CUDA_TRY(c, cudaMemcpyAsync(pl->Kh, Kh.data(), Kh.size() * sizeof(float), cudaMemcpyHostToDevice, c.stream));
  ASD_CUDA_TRY(c, cudaMemcpyAsync(pl->twx, twx.data(), twx.size() * sizeof(float2), cudaMemcpyHostToDevice, c.stream));
  ASD_CUDA_TRY(c, cudaMemcpyAsync(pl->twy, twy.data(), twy.size() * sizeof(float2), cudaMemcpyHostToDevice, c.stream));
  ASD_CUDA_TRY(c, cudaMemsetAsync(pl->B, 0, (size_t)3 * pl->dcx * pl->dcy * pl->dcz * sizeof(float), c.stream));
  ASD_CUDA_TRY(c, cudaMemsetAsync(pl->acc, 0, (size_t)3 * pl->dcx * pl->dcy * pl->dcz * sizeof(long long), c.stream));
  pl->acc_state = DemagPlan::ACC_CLEAN;
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));             // the host vectors are about to go out of scope
  graphs_invalidate(c);
  return ASD_OK;
}

// ---- stray field of the frozen track: workspace, enable, refresh ----
static int stray_xr(const Ctx& c, int range_cells) {
  const int far = (int)c.ncx - 1;
  return (range_cells > 0 && range_cells < far) ? range_cells : (far > 0 ? far : 0);
}
struct StrayCarve { size_t Nt, mom, Bt, total; };
static void stray_carve(const Ctx& c, const DemagPlan& pl, int XR, StrayCarve& cv) {
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes, 256); return o; };
  cv.Nt = take((size_t)(2 * XR + 1) * (2 * pl.dcy - 1) * (2 * pl.dcz - 1) * 6 * sizeof(float));
  cv.mom = take((size_t)c.ncell * 3 * sizeof(float));
  cv.Bt = take((size_t)3 * pl.dcx * pl.dcy * pl.dcz * sizeof(float));
  cv.total = off;
}
size_t demag_stray_workspace_bytes(Ctx& c, int range_cells) {
  if (!c.demag) return 0;
  StrayCarve cv;
  stray_carve(c, *c.demag, stray_xr(c, range_cells), cv);
  return cv.total;
}

// The field the frozen track adds to every window macrocell, for the current window origin and track state.
asd_status demag_stray_refresh(Ctx& c) {
  if (!c.demag || !c.demag->stray) return ASD_OK;
  DemagPlan& pl = *c.demag;
  const int mx = c.d.macro[0];
  const long long c0 = c.x0 / mx, c_last = (c.x0 + c.d.nx - 1) / mx;
  const long long cx_lo = std::max<long long>(0, c0 - pl.XR), cx_hi = std::min<long long>(c.ncx - 1, c_last + pl.XR);
  const long long n = (cx_hi - cx_lo + 1) * c.ncy * c.ncz;
  stray_moments_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c.stream>>>(
      c.col, c.out_sum, c.out_cnt, c.init_mean, pl.mom, cx_lo, cx_hi, (int)c.ncy, (int)c.ncz, mx, c.d.macro[1], c.d.macro[2],
      c.d.ny, c.d.nz, (long long)c.d.track_nx, (long long)c.x0, c.d.nx);
  ASD_LAUNCH_CHECK(c, "stray_moments");
  ASD_CUDA_TRY(c, cudaMemsetAsync(pl.Bt, 0, (size_t)3 * pl.dcx * pl.dcy * pl.dcz * sizeof(float), c.stream));
  const int ncw = (int)(c_last - c0 + 1);
  const int threads = std::min(1024, (int)align_up((size_t)(pl.dcy * pl.dcz), 32));
  stray_sum_kernel<<<(unsigned)ncw, threads, (size_t)c.ncy * c.ncz * 3 * sizeof(float), c.stream>>>(
      pl.Nt, pl.mom, pl.Bt, c0, cx_lo, cx_hi, pl.XR, pl.dcx, pl.dcy, pl.dcz, (int)c.ncy, (int)c.ncz);
  ASD_LAUNCH_CHECK(c, "stray_sum");
  c.demag_age = 0;                                              // a held cell field was made with the old stray field
  return ASD_OK;
}

asd_status demag_stray_enable(Ctx& c, int on, int range_cells, void* ws, size_t bytes) {
  DemagPlan& pl = *c.demag;
  if (!on) { pl.stray = false; c.demag_age = 0; return ASD_OK; }
  const int XR = stray_xr(c, range_cells);
  StrayCarve cv;
  stray_carve(c, pl, XR, cv);
  if (bytes < cv.total) { std::snprintf(c.err, sizeof(c.err), "asd_enable_track_stray: workspace too small"); return ASD_ENOMEM; }
  if ((size_t)c.ncy * c.ncz * 3 * sizeof(float) > 48 * 1024) {
    std::snprintf(c.err, sizeof(c.err), "asd_enable_track_stray: more than 4096 macrocells per track cross-section");
    return ASD_EUNSUPPORTED;
  }
  char* base = (char*)ws;
  pl.Nt = (float*)(base + cv.Nt); pl.mom = (float*)(base + cv.mom); pl.Bt = (float*)(base + cv.Bt);
  pl.XR = XR;
  // cuboid tensor for every source-target offset (fp64 on the host, as for the window's own field), times -mu_0 mu_s / V
  const int sy = 2 * pl.dcy - 1, sz = 2 * pl.dcz - 1;
  const double V = pl.cell[0] * pl.cell[1] * pl.cell[2], scale = -4.0e-7 * kPi * c.d.mu_s / V;
  std::vector<float> Nt((size_t)(2 * XR + 1) * sy * sz * 6);
  for (int a = -XR; a <= XR; ++a)
    for (int b = -(pl.dcy - 1); b <= pl.dcy - 1; ++b)
      for (int g = -(pl.dcz - 1); g <= pl.dcz - 1; ++g) {
        const double R[3] = {a * pl.cell[0], b * pl.cell[1], g * pl.cell[2]};
        double N[6];
        cuboid_tensor(pl.cell, R, N);
        float* dst = Nt.data() + (((size_t)(a + XR) * sy + (b + pl.dcy - 1)) * sz + (g + pl.dcz - 1)) * 6;
        for (int comp = 0; comp < 6; ++comp) dst[comp] = (float)(N[comp] * scale);
      }
  ASD_CUDA_TRY(c, cudaMemcpyAsync(pl.Nt, Nt.data(), Nt.size() * sizeof(float), cudaMemcpyHostToDevice, c.stream));
  ASD_CUDA_TRY(c, cudaMemsetAsync(pl.mom, 0, (size_t)c.ncell * 3 * sizeof(float), c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  pl.stray = true;
  return demag_stray_refresh(c);
}

// Host copy of the track's stray field per window macrocell (tests, diagnostics); synchronises.
asd_status demag_stray_field_host(Ctx& c, float* out) {
  DemagPlan& pl = *c.demag;
  const size_t cells = (size_t)pl.dcx * pl.dcy * pl.dcz;
  std::vector<float> h(3 * cells);
  ASD_CUDA_TRY(c, cudaMemcpyAsync(h.data(), pl.Bt, 3 * cells * sizeof(float), cudaMemcpyDeviceToHost, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  for (size_t q = 0; q < cells; ++q)
    for (int comp = 0; comp < 3; ++comp) out[3 * q + comp] = h[comp * cells + q];
  return ASD_OK;
}
bool demag_stray_on(const Ctx& c) { return c.demag && c.demag->stray; }

namespace {
template <typename... Args>
void launch_chain(void (*kern)(Args...), dim3 grid, unsigned threads, size_t smem, cudaStream_t stream, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  cudaLaunchKernelEx(&cfg, kern, args...);
}
}  // namespace

// Demagnetising field of the configuration in array block aX (S or S~) into demag->B, on c.launch_stream.
asd_status launch_demag(Ctx& c, int aX, bool may_use_acc) {
  DemagPlan& pl = *c.demag;
  long long* acc_used = nullptr;
  if (may_use_acc && pl.acc_state == DemagPlan::ACC_VALID && aX == c.aS) {
    // Eq. (6) was done by the corrector of the fused step that wrote these spins
    // latency-bound (one dependent load, one barrier, a 3 NKY x dcy transform): small CTAs so that all of them are
    // resident at once (two passes of row_ydft each)
    const unsigned threads = (unsigned)std::min<size_t>(1024, align_up((size_t)6 * pl.NKY, 32));
    launch_chain(cells_ydft, dim3((unsigned)(pl.dcx * pl.dcz)), threads, cg_smem_bytes(0, c.d.ny, pl), c.launch_stream,
                 (const long long*)pl.acc, (double)pl.mu_over_V / (double)pl.acc_fx, pl.dcx, pl.dcy, pl.dcz, pl.PY, pl.NKY,
                 (const float2*)pl.twy, pl.Y);
    ASD_LAUNCH_CHECK(c, "cells_ydft");
    acc_used = pl.acc;
    pl.acc_state = DemagPlan::ACC_CLEAN;
  } else {
    const int vec = (c.d.ny % 4 == 0) ? 4 : 1, groups = c.d.ny / vec;
    int lanes = 1024 / groups;
    if (lanes > kMaxRowLanes) lanes = kMaxRowLanes;
    if (const char* ev = std::getenv("ASD_CG_LANES")) { const int v = std::atoi(ev); if (v >= 1 && v <= lanes) lanes = v; }   // tuning override
    if (lanes < 1) lanes = 1;                                   // groups <= 1024 is checked at enable time
    const int threads = (int)align_up((size_t)(groups * lanes), 32);
    const size_t smem = cg_smem_bytes(lanes, c.d.ny, pl);
    const unsigned blocks = (unsigned)(pl.dcx * pl.dcz);
    launch_chain(vec == 4 ? coarse_grain_ydft<4> : coarse_grain_ydft<1>, dim3(blocks), (unsigned)threads, smem, c.launch_stream,
                 (const float*)c.arr(aX), (uint32_t)c.as, c.d.nx, c.d.ny, c.d.nz, c.nyp, c.lead, c.d.macro[0], c.d.macro[1],
                 c.d.macro[2], (long long)c.x0, pl.dcx, pl.dcy, pl.dcz, pl.PY, pl.NKY, pl.mu_over_V, lanes,
                 (const float2*)pl.twy, pl.Y);
    ASD_LAUNCH_CHECK(c, "coarse_grain_ydft");
  }
  launch_chain(demag_xconv, dim3((unsigned)pl.NKY, 3u), pl.xconv_threads, pl.xconv_smem, c.launch_stream,
               (const float2*)pl.Y, pl.Z, (const float*)pl.Kh, (const float2*)pl.twx, pl.dcx, pl.dcz, pl.PX, pl.logPX, pl.NKY,
               acc_used, 3 * pl.dcx * pl.dcy * pl.dcz);
  ASD_LAUNCH_CHECK(c, "demag_xconv");
  launch_chain(demag_yinv, dim3((unsigned)((pl.dcx + kYinvCols - 1) / kYinvCols), (unsigned)pl.F), 256u,
               ((size_t)pl.NKY * kYinvCols + pl.PY) * sizeof(float2), c.launch_stream,
               (const float2*)pl.Z, (const float2*)pl.twy, pl.B, pl.dcx, pl.dcy, pl.dcz, pl.PY, pl.NKY,
               (const float*)(pl.stray ? pl.Bt : nullptr));
  ASD_LAUNCH_CHECK(c, "demag_yinv");
  return ASD_OK;
}

long long* demag_acc_arm(Ctx& c, float& fx) {
  if (!c.demag) return nullptr;
  static const bool off = [] { const char* e = std::getenv("ASD_DEMAG_EPILOGUE"); return e && std::atoi(e) == 0; }();   // tuning override
  if (off) return nullptr;
  DemagPlan& pl = *c.demag;
  if (pl.acc_state != DemagPlan::ACC_CLEAN) {
    if (cudaMemsetAsync(pl.acc, 0, (size_t)3 * pl.dcx * pl.dcy * pl.dcz * sizeof(long long), c.launch_stream) != cudaSuccess) {
      cudaGetLastError();
      return nullptr;
    }
  }
  pl.acc_state = DemagPlan::ACC_VALID;
  fx = pl.acc_fx;
  return pl.acc;
}
void demag_acc_drop(Ctx& c) {
  if (c.demag && c.demag->acc_state == DemagPlan::ACC_VALID) c.demag->acc_state = DemagPlan::ACC_STALE;
}
void demag_held_invalidate(Ctx& c) {
  c.demag_age = 0;
  demag_acc_drop(c);
}

void demag_fill_params(const Ctx& c, StageParams& p) {
  p.dm.B = nullptr;
  if (!c.demag) return;
  const DemagPlan& pl = *c.demag;
  p.dm.B = pl.B;
  p.dm.comp_stride = (uint32_t)((size_t)pl.dcx * pl.dcy * pl.dcz);
  p.dm.sx = (uint32_t)(pl.dcy * pl.dcz); p.dm.sy = (uint32_t)pl.dcz;
  magic_u31((uint32_t)c.d.macro[0], p.dm.mx_m, p.dm.mx_s);
  magic_u31((uint32_t)c.d.macro[1], p.dm.my_m, p.dm.my_s);
  magic_u31((uint32_t)c.d.macro[2], p.dm.mz_m, p.dm.mz_s);
  p.dm.x0 = (uint32_t)c.x0; p.dm.c0 = (uint32_t)(c.x0 / c.d.macro[0]);
}

// Host copy of the cell field of the CURRENT spins (tests, diagnostics); synchronises.
asd_status demag_field_host(Ctx& c, float* out, int64_t dims[3], bool held) {
  DemagPlan& pl = *c.demag;
  dims[0] = pl.dcx; dims[1] = pl.dcy; dims[2] = pl.dcz;
  if (!out) return ASD_OK;
  c.launch_stream = c.stream;
  if (!held) {
    const asd_status st = launch_demag(c, c.aS);
    if (st != ASD_OK) return st;
  }
  const size_t cells = (size_t)pl.dcx * pl.dcy * pl.dcz;
  std::vector<float> h(3 * cells);
  ASD_CUDA_TRY(c, cudaMemcpyAsync(h.data(), pl.B, 3 * cells * sizeof(float), cudaMemcpyDeviceToHost, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  // cells of the spare x-slot that do not overlap the window at this alignment hold no site: reported as 0
  const int ncx = (int)((c.x0 + c.d.nx - 1) / c.d.macro[0] - c.x0 / c.d.macro[0]) + 1;
  for (int a = 0; a < pl.dcx; ++a)
    for (int b = 0; b < pl.dcy; ++b)
      for (int g = 0; g < pl.dcz; ++g)
        for (int comp = 0; comp < 3; ++comp)
          out[(((size_t)a * pl.dcy + b) * pl.dcz + g) * 3 + comp] =
              a < ncx ? h[comp * cells + ((size_t)a * pl.dcy + b) * pl.dcz + g] : 0.0f;
  return ASD_OK;
}

}  // namespace asd
