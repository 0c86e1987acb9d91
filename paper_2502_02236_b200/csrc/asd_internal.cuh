// asd_internal.cuh -- context, workspace layout and kernel parameter blocks of libasd (not part of the ABI).
//
// Device layout of every per-site array: "padded rows".
//   A row is the ny sites (i, k, 0..ny-1); rows are numbered r = i*nz + k, so x is slowest and a window shift is
//   one contiguous move.  Each row is stored with stride nyp = round_up(ny, 4) + 4 floats; the nyp - ny trailing
//   floats are zero for ever.  lead = nyp + 4 zero floats precede row 0.  Element of site (r, j):  e = lead + r*nyp + j.
//   => the y-1 neighbour of j = 0 and the y+1 neighbour of j = ny-1 are zeros that sit next to the row in memory,
//      and a missing x+-1 / z+-1 row is read from the zero lead (at element j + 4, so that its j-1 and j+4 edge
//      reads stay inside the lead): open boundaries cost no predicate and no mask,
//      and 128-bit loads stay aligned (nyp % 4 == 0).
//   The 13 per-site arrays (S, S~, A: 3 components each; sigma; B: 3) are consecutive with one stride `as`
//   (elements), so one 32-bit element offset addresses all of them.
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
  BOND_ALL_XP = BOND_XP | BOND_XPYP | BOND_XPYM, BOND_ALL_XM = BOND_XM | BOND_XMYP | BOND_XMYM,
  // bit 24: the 4-aligned group of columns (gx, 4q .. 4q+3) this column belongs to holds two DIFFERENT grains (the film
  // kernel then gathers anisotropy parameters per site instead of once per group)
  COL_GROUP_MIXED = 1u << 24
};

// indices of the 13 per-site arrays inside the block `arrays` (stride `as` elements)
enum : int { AR_S = 0, AR_ST = 3, AR_A = 6, AR_SIGMA = 9, AR_B = 10, AR_COUNT = 13 };

struct Vec3Ptr { float *x, *y, *z; };
struct CVec3Ptr { const float *x, *y, *z; };

// n / d for n < 2^31 by multiply-high (m == 0 means d == 1): m = floor(2^(31+L)/d) + 1, s = L - 1, L = ceil(log2 d)
// (Granlund-Montgomery round-up method with 31-bit dividends: exact).
inline void magic_u31(uint32_t d, uint32_t& m, uint32_t& s) {
  if (d <= 1) { m = 0; s = 0; return; }
  uint32_t L = 0;
  while ((1ull << L) < d) ++L;
  m = (uint32_t)(((1ull << (31 + L)) / d) + 1ull);
  s = L - 1;
}

// Where a stage kernel finds the demagnetising field of a site's macrocell (asd_demag.cu):
//   B[comp * comp_stride + ci * sx + cj * sy + ck],  ci = (x0 + i) / mx - c0,  cj = j / my,  ck = k / mz
// with the three divisions done by multiply-high (magic_u31).
struct DemagGeom {
  const float* B;              // nullptr = demag off
  uint32_t comp_stride, sx, sy;
  uint32_t mx_m, mx_s, my_m, my_s, mz_m, mz_s;
  uint32_t x0, c0;
};
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t div_u31(uint32_t n, uint32_t m, uint32_t s) { return m ? (__umulhi(n, m) >> s) : n; }
// offset of the macrocell of window site (i, j, k) inside one component of dm.B
__device__ __forceinline__ uint32_t demag_cell(const DemagGeom& dm, uint32_t i, uint32_t j, uint32_t k) {
  return (div_u31(dm.x0 + i, dm.mx_m, dm.mx_s) - dm.c0) * dm.sx + div_u31(j, dm.my_m, dm.my_s) * dm.sy +
         div_u31(k, dm.mz_m, dm.mz_s);
}
__device__ __forceinline__ void demag_at(const DemagGeom& dm, uint32_t i, uint32_t j, uint32_t k, float Bd[3]) {
  const uint32_t q = demag_cell(dm, i, j, k);
  Bd[0] = __ldg(dm.B + q); Bd[1] = __ldg(dm.B + (dm.comp_stride + q)); Bd[2] = __ldg(dm.B + (2u * dm.comp_stride + q));
}
#endif

// Device copy of the two values that change between replays of a captured CUDA graph: the step index and the
// head-field scale.  A kernel launched with dyn != nullptr takes step = dyn step + its own n_lo (its offset inside
// the graph) and the scale from here instead of from its (frozen) parameter block.
struct DynState { uint32_t n_lo, n_hi; float scale; uint32_t pad; };
#ifdef __CUDACC__
__device__ __forceinline__ void resolve_dyn(const DynState* dyn, uint32_t& n_lo, uint32_t& n_hi, float& scale) {
  if (dyn) {
    const uint64_t n = (((uint64_t)dyn->n_hi << 32) | dyn->n_lo) + n_lo;
    n_lo = (uint32_t)n; n_hi = (uint32_t)(n >> 32); scale = dyn->scale;
  }
}
#endif

// Parameters of one Heun stage (passed by value; lives in the constant bank).
struct StageParams {
  float* arrays;               // base of the 13 padded per-site arrays
  uint32_t as;                 // array stride, elements
  uint32_t aX, aA, aOut, aOutA;  // array index (AR_*) of: the configuration whose neighbours are read (S or S~),
                               // A = S + dt/2 k1 (corrector input), the output spins, the A output (predictor)
  const uint32_t* col;         // column table at the window origin: col[i*ny + j]
  const float4* grain;         // (e_x, e_y, e_z, 2 k_u / mu_s) per grain id + 1 (entry 0 = vacant: zeros)
  const float* aniso;          // per-column SoA copy of the same: e_x | e_y | e_z | 2k_u/mu_s, each [track_nx*ny],
  uint32_t aniso_stride;       //   at the window origin; component stride in elements
  const int32_t* ell_idx;      // general ELL, slot-major [W][N]: padded element offset of the neighbour; an empty slot
                               // holds the site itself with J = 0 (ell_transpose_kernel), never -1
  const float* ell_J;          // J_ij / mu_s [Tesla], slot-major
  int32_t ell_w;
  int32_t nx, ny, nz, nyp;     // nyp = padded row stride
  int32_t lead;                // zero floats before row 0 (nyp + 4)
  uint32_t nrows, ngrp;        // nx*nz; threads per row
  uint32_t nthreads;           // nrows * ngrp
  uint32_t N;                  // nx*ny*nz (dense count; < 2^31)
  int32_t pbc_x, pbc_y, pbc_z;
  float jx[3];                 // J_shell / mu_s [Tesla]
  float gdt;                   // gamma dt / (1 + lambda^2)
  float lambda;
  float scale;                 // B_app = scale * B
  uint32_t n_lo, n_hi;         // step index before the step (with dyn: offset of this step inside the graph)
  const DynState* dyn;         // nullptr outside graph replays
  DemagGeom dm;                // demagnetising field per macrocell (asd_demag.cu); dm.B == nullptr: off
  const float* edgeB;          // multiscale window (asd_mm.cu): exchange field of the held mesh directions on the sites of
                               // plane 0 (side 0) and nx-1 (side 1), [side][component][nz*nyp] padded rows; nullptr: off
  uint64_t g0;                 // x0 * ny * nz: global id of window site 0
  PhiloxKey key;
};


struct DemagPlan;           // asd_demag.cu: plans, transformed tensor and buffers of the demagnetising field
struct TmaPlan;             // asd_heun_tma.cu: tensor maps + strip / chunk plan of the staged film kernel
struct FusedPlan;           // asd_heun_fused.cu: tensor map + strip / chunk plan of the one-kernel Heun step
struct MmPlan;              // asd_mm.cu: the micromagnetic meshes of the multiscale window

struct Ctx {
  asd_lattice_desc d;          // host pointers inside are NOT valid after create
  cudaStream_t stream = nullptr;
  cudaStream_t launch_stream = nullptr;   // where the stage kernels go: `stream`, or the capture stream while a graph is recorded
  int device = 0;
  int sm_count = 148;
  int64_t N = 0;               // dense sites
  int32_t nyp = 0;             // padded row stride
  int32_t lead = 0;            // zero floats before row 0
  int64_t nrows = 0;           // nx*nz
  int64_t Np = 0;              // elements of one padded array: lead + nrows*nyp
  int64_t as = 0;              // array stride (elements)
  int32_t plane = 0;           // dense ny*nz
  double gamma = 0;
  // device arrays (sub-allocated from the caller's workspace)
  float* arrays = nullptr;
  int aS = AR_S, aSt = AR_ST;  // which third of the spin block currently holds S / the scratch S~ (swapped by a shift)
  uint32_t *col = nullptr;          // [track_nx * ny]
  int32_t *grain_map_dev = nullptr; // [track_nx * ny] as given
  float4 *grain = nullptr;          // [n_grains + 1]
  float *aniso = nullptr;           // [4][track_nx * ny]
  int32_t *flags = nullptr;         // [16] device: flags[0] = 1 if two different grains touch; flags[4..7] = DynState
  int32_t *ell_idx = nullptr; float *ell_J = nullptr;
  bool grains_touch = true;
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
  long long *grain_scratch = nullptr;   // pinned, [n_grains*4]: asd_grain_magnetisation's device-to-host landing area
  // state
  float scale = 1.0f;
  int64_t step = 0, shift = 0, pass = 0, x0 = 0;
  int32_t kernel_variant = ASD_KERNEL_AUTO;
  // CUDA-graph replay of asd_step_heun(n) (asd_graph.cu)
  int32_t graph_mode = ASD_GRAPH_AUTO;
  cudaStream_t cap_stream = nullptr;   // internal stream the graphs are captured on (the caller's may be the legacy one)
  struct GraphCache* graphs = nullptr;
  // double-buffered field upload (asd_stage_fields_host / asd_commit_fields): caller-owned staging of 4 dense arrays
  float* staging = nullptr;
  cudaStream_t copy_stream = nullptr;   // the H2D copies run here, beside the stage kernels on `stream`
  cudaEvent_t staged_ev = nullptr, consumed_ev = nullptr;
  uint32_t staged_mask = 0;             // bit a: array a (T, Bx, By, Bz) was staged and awaits asd_commit_fields
  DemagPlan* demag = nullptr;       // non-null once asd_enable_demag succeeded
  int32_t demag_every = 0;          // 0: field recomputed in every stage; P >= 1: from S at every P-th Heun step, held in between
  int64_t demag_age = 0;            // Heun steps since the held field was last invalidated (enable, shift, set_spins)
  int32_t demag_refresh = 3;        // this step: bit 0 = recompute before the predictor, bit 1 = before the corrector
  MmPlan* mm = nullptr;             // non-null once asd_mm_enable succeeded
  // window ends exchange coupled to the frozen track (asd_enable_track_exchange; reading E1): the track's
  // directions beyond the two ends and the edge field they make on planes 0 / nx-1 (caller's workspace)
  bool tex_on = false;
  float* tex_ghost = nullptr;       // [2][3][ncy*ncz]
  float* tex_edgeB = nullptr;       // [2][3][nz*nyp]
  TmaPlan* tma_plan = nullptr;      // built lazily by the first staged launch (host memory, freed by asd_destroy)
  bool tma_plan_tried = false;
  FusedPlan* fused_plan = nullptr;  // likewise for the fused one-kernel step
  bool fused_plan_tried = false;
  int64_t launches = 0;
  bool cuda_failed = false;
  char err[256] = {0};

  float* arr(int a) const { return arrays + (size_t)a * (size_t)as; }
  Vec3Ptr vec(int a) const { return Vec3Ptr{arr(a), arr(a + 1), arr(a + 2)}; }
  Vec3Ptr S() const { return vec(aS); }
  Vec3Ptr St() const { return vec(aSt); }
  Vec3Ptr A() const { return vec(AR_A); }
  float* sigma() const { return arr(AR_SIGMA); }
  float* B(int c) const { return arr(AR_B + c); }
  const uint32_t* col_win() const { return col + x0 * d.ny; }
};

constexpr int kMaxPartialBlocks = 1024;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Workspace layout: one place computes every offset (used by asd_workspace_bytes and asd_create_lattice).
struct Layout {
  size_t arrays, col, gmap, grain, aniso, flags, ell_idx, ell_J, init_mean, cell_frame, out_sum, out_cnt,
      partials, grain_acc, total;
  int64_t N, nrows, Np, as, ncx, ncy, ncz, ncell;
  int32_t nyp, lead;
};
bool compute_layout(const asd_lattice_desc& d, Layout& L);
bool validate_desc(const asd_lattice_desc* d, const char** why);

// kernels / launchers (defined in the .cu files)
asd_status launch_build_columns(Ctx& c);
asd_status launch_pack_spins(Ctx& c, CVec3Ptr dense_src /* null members: +z */, Vec3Ptr padded_dst);
asd_status launch_unpack(Ctx& c, const float* padded, float* dense);
asd_status launch_pack_field(Ctx& c, const float* dense, float* padded);
asd_status launch_sigma(Ctx& c, const float* T_dense);
asd_status launch_heun(Ctx& c, int64_t n);                    // n Heun steps, through graphs when enabled
asd_status launch_heun_direct(Ctx& c, int64_t n, const DynState* dyn);   // 2n plain launches on c.stream (or the capture stream)
void graphs_invalidate(Ctx& c);                               // drop cached graphs (after a shift / a kernel change)
void graphs_free(Ctx& c);
DynState* dyn_state(const Ctx& c);
// demagnetising field (asd_demag.cu)
size_t demag_workspace_bytes(Ctx& c);
asd_status demag_enable(Ctx& c, const double spacing[3], void* ws, size_t bytes);
void demag_free(Ctx& c);
asd_status launch_demag(Ctx& c, int aX, bool may_use_acc = false);   // field of the configuration in arrays aX..aX+2
// Eq. (6) folded into the fused step's corrector: the macrocell sums of the spins a step writes, as 64-bit fixed point
long long* demag_acc_arm(Ctx& c, float& fx);                  // zeroed buffer for the step about to be launched (or nullptr), its scale
void demag_acc_drop(Ctx& c);                                  // the spins changed by other means: the sums are stale
void demag_held_invalidate(Ctx& c);                           // ... and so is the held field (age 0)
void demag_fill_params(const Ctx& c, StageParams& p);
asd_status demag_field_host(Ctx& c, float* out, int64_t dims[3], bool held = false);   // held: the stored field, nothing recomputed
size_t demag_stray_workspace_bytes(Ctx& c, int range_cells);     // stray field of the frozen track (reading D4)
asd_status demag_stray_enable(Ctx& c, int on, int range_cells, void* ws, size_t bytes);
asd_status demag_stray_refresh(Ctx& c);                          // after the window origin or the track store changed
asd_status demag_stray_field_host(Ctx& c, float* out);
bool demag_stray_on(const Ctx& c);
asd_status launch_heun_fast(Ctx& c, StageParams& p);          // one Heun step (2 kernels), fast path
bool heun_fast_supported(const Ctx& c);
asd_status launch_heun_ell(Ctx& c, StageParams& p);           // one Heun step (2 kernels), general ELL table
bool heun_ell_supported(const Ctx& c);
asd_status launch_heun_tma(Ctx& c, StageParams& p);           // one Heun step (2 kernels), TMA-staged film path
bool heun_tma_supported(const Ctx& c);
TmaPlan* tma_plan(Ctx& c);                                    // nullptr if the plan cannot be built
void tma_plan_free(Ctx& c);
asd_status launch_heun_fused(Ctx& c, StageParams& p);         // one Heun step (1 kernel); swaps the roles of the spin buffers
bool heun_fused_supported(const Ctx& c);
bool heun_fused_preferred(Ctx& c);                            // what ASD_KERNEL_AUTO asks (builds the plan)
FusedPlan* fused_plan(Ctx& c);
bool heun_fused_takes_mm(Ctx& c);                             // the plan's CTA shape has a multiscale instance
bool heun_fused_takes_demag(Ctx& c, bool with_edge_field = false);                          // ... a held-demagnetising-field instance
asd_status launch_heun_persist(Ctx& c, StageParams& p, int64_t n);   // n Heun steps in one cluster launch (asd_heun_persist.cu)
bool heun_persist_supported(const Ctx& c);
bool heun_persist_preferred(const Ctx& c);                    // what ASD_KERNEL_AUTO asks (measured crossover vs graph replay)
void fused_plan_free(Ctx& c);
void fill_stage_params(const Ctx& c, StageParams& p);
// multiscale window (asd_mm.cu)
size_t mm_workspace_bytes(const Ctx& c, const int32_t mcx[2]);
asd_status mm_enable(Ctx& c, const asd_mm_desc& d, void* ws, size_t bytes);
void mm_free(Ctx& c);
asd_status mm_before_step(Ctx& c);                            // exchange + RK4 step when the cadence says so
void mm_restart_cadence(Ctx& c);
const float* mm_edge_field(const Ctx& c);                       // the meshes' edge field, else the track's, else nullptr
inline bool edge_field_on(const Ctx& c) { return c.mm != nullptr || c.tex_on; }
size_t track_exchange_workspace_bytes(const Ctx& c);
asd_status track_exchange_enable(Ctx& c, int on, void* ws, size_t bytes);
asd_status track_exchange_refresh(Ctx& c);                      // after the window origin or the track store changed
asd_status mm_set_fields_host(Ctx& c, int side, const float* T, const float* Bx, const float* By, const float* Bz);
asd_status mm_set_m_host(Ctx& c, int side, const float* m);
asd_status mm_get_m_host(Ctx& c, int side, float* m);
void mm_dims(const Ctx& c, int side, int64_t dims[3]);
asd_status mm_shift_prepare(Ctx& c, int pc);
const float* mm_shift_frames(const Ctx& c);
asd_status mm_shift_finish(Ctx& c, int pc);
asd_status mm_flush_to_track(Ctx& c);                         // end of a pass: every mesh cell -> track store
asd_status mm_restart_from_track(Ctx& c);                     // start of a pass: meshes along the track under them
asd_status launch_shift_mm(Ctx& c, int32_t p);                // asd_shift.cu: whole-cell shift of a multiscale window
asd_status launch_shift(Ctx& c, int32_t p);
asd_status launch_cell_frames(Ctx& c);
asd_status launch_track_end_pass(Ctx& c);
asd_status launch_track_begin_pass(Ctx& c, int64_t x0_new);
asd_status launch_track_read_scan(Ctx& c, double y_r, double sigma_x, double sigma_y, double x_first, double x_step,
                                  int64_t count, double* out_host);
asd_status launch_magnetisation(Ctx& c, double out4[4], int32_t i0 = -1, int32_t n = 0);   // i0 < 0: the whole window
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

#ifdef __CUDACC__
namespace asd {
// Launch with programmatic stream serialization (programmatic dependent launch): the grid may be scheduled before its
// predecessor in the stream has finished and synchronises with it at its own griddepcontrol.wait.
template <class Params>
inline void launch_pdl(void (*kern)(const Params), unsigned blocks, unsigned threads, cudaStream_t stream, const Params& p,
                       bool allow = true) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(blocks); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = 0; cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = allow ? 1 : 0;             // recorded graphs keep plain edges (measured faster there)
  cudaLaunchKernelEx(&cfg, kern, p);
}
}  // namespace asd
#endif

struct asd_ctx { asd::Ctx c; };
