// asd_internal.cuh -- context, workspace layout and kernel parameter blocks of libasd (not part of the ABI).
#pragma once
#include <cstddef>
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

#include "../../include/asd.h"
#include "asd_rng.cuh"

namespace asd {

constexpr double kBoltzmann = 1.380649e-23;        // J/K
constexpr double kGammaDefault = 1.76085963023e11; // rad s^-1 T^-1 (Q3)

// Column table entry (one per track column (gx, j), shared by the nz sites of the column):
//   bits 0..15  grain id + 1 (0 = vacant column)
//   bits 16..23 in-plane bond mask: a bond exists iff the neighbour column exists (open edge in y, or the
//               track end in x), is magnetic and belongs to the SAME grain (P:29 exchange-decoupled grains).
// Window edges in x (open boundary) are applied in the kernels, so the table does not change on a shift.
enum : uint32_t {
  BOND_XP = 1u << 16, BOND_XM = 1u << 17, BOND_YP = 1u << 18, BOND_YM = 1u << 19,
  BOND_XPYP = 1u << 20, BOND_XPYM = 1u << 21, BOND_XMYP = 1u << 22, BOND_XMYM = 1u << 23,
  BOND_ALL_XP = BOND_XP | BOND_XPYP | BOND_XPYM, BOND_ALL_XM = BOND_XM | BOND_XMYP | BOND_XMYM
};

struct Vec3Ptr { float *x, *y, *z; };
struct CVec3Ptr { const float *x, *y, *z; };

// Parameters of one Heun stage (passed by value; lives in the constant bank).
struct StageParams {
  CVec3Ptr X;        // configuration whose neighbours are read: S (predictor) or S~ (corrector)
  CVec3Ptr A;        // corrector only: A = S + dt/2 k1 of the own site
  Vec3Ptr out;       // predictor: S~ ; corrector: new S
  Vec3Ptr outA;      // predictor only: A
  const float *sigma;          // c_th sqrt(T_i)  [Tesla]
  const float *Bx, *By, *Bz;   // applied field [Tesla]
  const uint32_t *col;         // column table at the window origin: col[i*ny + j]
  const float4 *grain;         // (e_x, e_y, e_z, 2 k_u / mu_s) per grain
  const int32_t *ell_idx;      // general ELL, slot-major [W][N] (or null)
  const float *ell_J;          // J_ij / mu_s [Tesla], slot-major
  int32_t ell_w;
  int32_t nx, ny, nz, plane;   // plane = ny*nz
  int64_t N;
  int32_t pbc_x, pbc_y, pbc_z;
  float jx[3];                 // J_shell / mu_s [Tesla]
  float gdt;                   // gamma dt / (1 + lambda^2)
  float lambda;
  float scale;                 // B_app = scale * B
  uint32_t n_lo, n_hi;         // step index before the step
  uint64_t g0;                 // x0 * plane: global id of window site 0
  PhiloxKey key;
};

struct Ctx {
  asd_lattice_desc d;          // host pointers inside are NOT valid after create
  cudaStream_t stream = nullptr;
  int device = 0;
  int sm_count = 148;
  int64_t N = 0, Npad = 0;
  int32_t plane = 0;
  double gamma = 0;
  // device arrays (sub-allocated from the caller's workspace)
  Vec3Ptr S{}, St{}, A{};
  float *sigma = nullptr, *Bx = nullptr, *By = nullptr, *Bz = nullptr;
  uint32_t *col = nullptr;          // [track_nx * ny]
  int32_t *grain_map_dev = nullptr; // [track_nx * ny] as given
  float4 *grain = nullptr;          // [n_grains]
  int32_t *ell_idx = nullptr; float *ell_J = nullptr;
  // track store
  int64_t ncx = 0, ncy = 0, ncz = 0, ncell = 0;
  float *init_mean = nullptr;       // [ncell*3]
  float *cell_frame = nullptr;      // [ncell*12]: theta_max, n(3), e1(3), e2(3), pad(2)
  double *out_sum = nullptr;        // [ncell*3]
  long long *out_cnt = nullptr;     // [ncell]
  // reductions
  double *partials = nullptr;       // [kMaxPartialBlocks*4]
  long long *grain_acc = nullptr;   // [n_grains*4] fixed-point sums and counts
  double *host_scratch = nullptr;   // pinned, 4 doubles
  // state
  float scale = 1.0f;
  int64_t step = 0, shift = 0, pass = 0, x0 = 0;
  int32_t kernel_variant = ASD_KERNEL_AUTO;
  int64_t launches = 0;
  bool cuda_failed = false;
  char err[256] = {0};
};

constexpr int kMaxPartialBlocks = 1024;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Workspace layout: one place computes every offset (used by asd_workspace_bytes and asd_create_lattice).
struct Layout {
  size_t spins[9], sigma, B[3], col, gmap, grain, ell_idx, ell_J, init_mean, cell_frame, out_sum, out_cnt,
      partials, grain_acc, total;
  int64_t N, Npad, ncx, ncy, ncz, ncell;
};
bool compute_layout(const asd_lattice_desc& d, Layout& L);
bool validate_desc(const asd_lattice_desc* d, const char** why);

// kernels / launchers (defined in the .cu files)
asd_status launch_build_columns(Ctx& c);
asd_status launch_init_spins(Ctx& c);
asd_status launch_mask_spins(Ctx& c, CVec3Ptr src, Vec3Ptr dst);
asd_status launch_sigma(Ctx& c, const float* T_dev);
asd_status launch_heun(Ctx& c, int64_t n);
asd_status launch_shift(Ctx& c, int32_t p);
asd_status launch_cell_frames(Ctx& c);
asd_status launch_magnetisation(Ctx& c, double out4[4]);
asd_status launch_grain_magnetisation(Ctx& c, double* m_host);
asd_status launch_ell_transpose(Ctx& c, const int32_t* idx_site_major, const float* J_site_major);

asd_status fail_cuda(Ctx& c, cudaError_t e, const char* where);
#define ASD_CUDA_TRY(ctx, expr)                                         \
  do {                                                                  \
    cudaError_t e__ = (expr);                                           \
    if (e__ != cudaSuccess) return ::asd::fail_cuda((ctx), e__, #expr); \
  } while (0)
#define ASD_LAUNCH_CHECK(ctx, name)                                     \
  do {                                                                  \
    (ctx).launches += 1;                                                \
    cudaError_t e__ = cudaGetLastError();                               \
    if (e__ != cudaSuccess) return ::asd::fail_cuda((ctx), e__, name);  \
  } while (0)

}  // namespace asd

struct asd_ctx { asd::Ctx c; };
