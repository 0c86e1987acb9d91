// asd_heun_tma.cu -- the hot path, staged film variant: one fused kernel per stochastic-Heun stage in which the
// spin planes are staged in shared memory by the TMA (cp.async.bulk.tensor) behind an mbarrier ring.
//
// Same lattices as asd_heun_fast.cu (open boundaries, built-in shells, ny % 4 == 0, grains that do not touch), same
// arithmetic per site (asd_site.cuh), same bytes to and from HBM (52 per site per stage).  What
// differs is how the bytes move:
//   * The window is cut into y-strips of BY sites and x-chunks of CX planes; one CTA owns one (strip, chunk) and
//     MARCHES along x through its chunk.  A thread owns 4 consecutive y-sites of one z-row of the strip and keeps
//     that (row, y-group) for the whole march, so nothing is re-derived per plane.
//   * The configuration X (S in the predictor, S~ in the corrector) is needed by the site itself and by its
//     neighbours.  One TMA instruction per plane brings the box [3 components] x [nz + 2 rows] x [BY + 8 sites] of
//     plane i+2 into a 4-slot ring while plane i is being computed from slots i-1, i, i+1: every plane is fetched
//     once per CTA, 2 planes ahead, with no registers tied up.  Out-of-range coordinates (y = -1, y = ny, z = -1,
//     z = nz, x = -1, x = nx) are zero-filled by the TMA, which IS the open boundary condition of Eq. (2)
//     (a missing neighbour contributes J * 0) -- no predicate, no mask, no padded copy.
//   * The per-column anisotropy parameters (e_x, e_y, e_z, 2 k_u/mu_s) of the strip ride on the same barrier.
//   * sigma, B (and A in the corrector) are read by exactly one thread each: they stream straight into registers
//     with 128-bit no-allocate loads issued at the top of the plane, and are consumed after the exchange sums and
//     the Philox / Box-Muller phase, which hides their latency.
//   * Results leave with 128-bit stores.
#include <cuda.h>

#include <cstdlib>

#include "asd_internal.cuh"
#include "asd_site.cuh"
#include "asd_tma.cuh"

namespace asd {

namespace {

constexpr int LAT_SC = 0, LAT_L10 = 1;
constexpr int kSlots = 4;          // ring of X planes: i-1, i, i+1 in use, i+2 in flight

struct TmaParams {
  const float* arrays;
  float* arrays_w;
  uint32_t as;                     // array stride (elements)
  int32_t aX;                      // array index of component 0 of the configuration read through the TMA
  uint32_t oA, oOut, oOutA, oSigma, oB;   // element offsets (array index * as)
  int32_t nx, ny, nz, nyp, lead;
  int32_t BY, G, nstrips, CX;      // strip width (sites), y-groups per strip row (BY / 4), strips, planes per chunk
  int32_t x0;                      // global plane of window plane 0 (anisotropy table coordinate)
  uint32_t main_pitch, edge_pitch; // shared-memory bytes reserved for the main box / one edge box (multiples of 128)
  uint32_t an_pitch;               // ... for one anisotropy box
  float j1, j2, j3;
  float gdt, lambda, scale;
  uint32_t n_lo, n_hi;
  const DynState* dyn;
  uint64_t g0;
  PhiloxKey key;
};

// Shared memory: [kSlots "full" + kSlots "empty" mbarriers, padded to 128 B][kSlots plane slots][2 anisotropy boxes].
// A plane slot holds three TMA boxes of one X plane, each float [3 components][nz + 2 rows (z = -1 .. nz)][w]:
//   main box   w = BY : the strip's own columns y = j0 .. j0+BY-1.  Its rows are CONTIGUOUS (no halo inside a row), so
//                       thread t reads the 16-byte unit t + const of the box: conflict-free for any strip width;
//   left edge  w = 4  : y = j0-4 .. j0-1   (only column j0-1 is used: the y-1 neighbour of the strip's first site);
//   right edge w = 4  : y = j0+BY .. j0+BY+3 (only column j0+BY is used).
// A thread's y-1 / y+4 neighbour lives in the main box unless the thread owns the first / last group of a row.
template <int LAT, int STAGE, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
heun_stage_tma(const __grid_constant__ CUtensorMap mapMain, const __grid_constant__ CUtensorMap mapEdge,
               const __grid_constant__ CUtensorMap mapAn, const TmaParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const uint32_t sm0 = smem_u32(smem_raw);
  const uint32_t bar_full = sm0, bar_empty = sm0 + 8u * kSlots;
  const uint32_t slot_pitch = p.main_pitch + 2u * p.edge_pitch;
  const uint32_t slots = sm0 + 128u;
  const uint32_t anbox = slots + kSlots * slot_pitch;

  const int tid = (int)threadIdx.x;
  const int strip = (int)blockIdx.x % p.nstrips, chunk = (int)blockIdx.x / p.nstrips;
  const int j0 = strip * p.BY;
  const int i_begin = chunk * p.CX;
  const int L = min(p.CX, p.nx - i_begin);            // planes of this CTA
  const uint32_t main_bytes = (uint32_t)(3 * (p.nz + 2) * p.BY * 4), edge_bytes = (uint32_t)(3 * (p.nz + 2) * 16);

  // plane m of the march (m = 0 is window plane i_begin - 1, the trailing halo) -> slot m % kSlots; the anisotropy
  // box of march step n = m - 2 rides on the same barrier.
  auto issue = [&](int m) {
    const uint32_t s = (uint32_t)(m & (kSlots - 1));
    const uint32_t bar = bar_full + 8u * s;
    const int n = m - 2;
    const bool with_an = (n >= 0 && n < L);
    mbar_expect_tx(bar, main_bytes + 2u * edge_bytes + (with_an ? (uint32_t)(16 * p.BY) : 0u));
    const uint32_t dst = slots + s * slot_pitch;
    const int xi = i_begin - 1 + m;
    tma_load_4d(dst, &mapMain, bar, j0, -1, xi, p.aX);
    tma_load_4d(dst + p.main_pitch, &mapEdge, bar, j0 - 4, -1, xi, p.aX);
    tma_load_4d(dst + p.main_pitch + p.edge_pitch, &mapEdge, bar, j0 + p.BY, -1, xi, p.aX);
    if (with_an) tma_load_3d(anbox + (uint32_t)(n & 1) * p.an_pitch, &mapAn, bar, j0, p.x0 + i_begin + n, 0);
  };

  if (tid == 0) {
    for (int s = 0; s < kSlots; ++s) { mbar_init(bar_full + 8u * s, 1u); mbar_init(bar_empty + 8u * s, (uint32_t)(NT / 32)); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (int m = 0; m < kSlots && m <= L + 1; ++m) issue(m);
  }
  __syncthreads();

  // ---- this thread's (row, y-group): fixed for the whole march ----
  const int k = tid / p.G, g = tid - k * p.G;
  const int j = j0 + 4 * g;
  const bool active = (k < p.nz) && (j < p.ny);
  // byte offsets inside a slot (component 0).  Row k+1 of a box is z = k (row 0 is z = -1).
  const uint32_t comp_main = (uint32_t)((p.nz + 2) * p.BY * 4), comp_edge = (uint32_t)((p.nz + 2) * 16);
  const uint32_t row_b = (uint32_t)(p.BY * 4);
  const uint32_t own_b = (uint32_t)(((k + 1) * p.BY + 4 * g) * 4);
  const bool first = (g == 0), last = (g == p.G - 1);
  const uint32_t left_b = first ? p.main_pitch + (uint32_t)((k + 1) * 16 + 12) : own_b - 4u;
  const uint32_t right_b = last ? p.main_pitch + p.edge_pitch + (uint32_t)((k + 1) * 16) : own_b + 16u;
  const uint32_t left_c = first ? comp_edge : comp_main, right_c = last ? comp_edge : comp_main;
  uint32_t e = (uint32_t)(p.lead + (i_begin * p.nz + k) * p.nyp + j);      // padded element of the first own site
  const uint32_t planep = (uint32_t)(p.nz * p.nyp);
  uint64_t gsite = p.g0 + (uint64_t)((uint32_t)(i_begin * p.nz + k) * (uint32_t)p.ny + (uint32_t)j);
  const uint32_t gplane = (uint32_t)(p.nz * p.ny);
  uint32_t n_lo = p.n_lo, n_hi = p.n_hi; float scale = p.scale;
  resolve_dyn(p.dyn, n_lo, n_hi, scale);
  const SiteConst sc{p.gdt, p.lambda, scale};

  mbar_wait(bar_full + 0u, 0u);
  mbar_wait(bar_full + 8u, 0u);

  for (int n = 0; n < L; ++n) {
    // streaming inputs of this plane: issued first, used last
    float4 sg4, bx4, by4, bz4, a4[3];
    if (active) {
      sg4 = ldg_stream4(p.arrays + (p.oSigma + e));
      bx4 = ldg_stream4(p.arrays + (p.oB + e));
      by4 = ldg_stream4(p.arrays + (p.oB + p.as + e));
      bz4 = ldg_stream4(p.arrays + (p.oB + 2u * p.as + e));
      if (STAGE == 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c) a4[c] = ldg_stream4(p.arrays + (p.oA + (uint32_t)c * p.as + e));
      }
    }
    {
      const int m = n + 2;                                   // plane i + 1 (and this step's anisotropy box)
      mbar_wait(bar_full + 8u * (uint32_t)(m & (kSlots - 1)), (uint32_t)(m >> 2) & 1u);
    }
    if (active) {
      const uint32_t prev = slots + (uint32_t)(n & (kSlots - 1)) * slot_pitch;
      const uint32_t cur = slots + (uint32_t)((n + 1) & (kSlots - 1)) * slot_pitch;
      const uint32_t next = slots + (uint32_t)((n + 2) & (kSlots - 1)) * slot_pitch;

      // ---- exchange field, Eq. (2): shell sums first, one multiply per shell ----
      float own[3][6];                // own row with its y-1 and y+1 edge sites
      float Bex[3][4];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const uint32_t cm = (uint32_t)c * comp_main, cl = (uint32_t)c * left_c, cr = (uint32_t)c * right_c;
        const float4 o = lds4(cur + own_b + cm);
        own[c][0] = lds1(cur + left_b + cl); own[c][1] = o.x; own[c][2] = o.y; own[c][3] = o.z; own[c][4] = o.w;
        own[c][5] = lds1(cur + right_b + cr);
        const float4 zp = lds4(cur + own_b + cm + row_b), zm = lds4(cur + own_b + cm - row_b);
        const float4 xp = lds4(next + own_b + cm), xm = lds4(prev + own_b + cm);
        const float zs[4] = {zp.x + zm.x, zp.y + zm.y, zp.z + zm.z, zp.w + zm.w};
        if (LAT == LAT_SC) {
          // 6 nearest neighbours, one J
          const float xs[4] = {xp.x + xm.x, xp.y + xm.y, xp.z + xm.z, xp.w + xm.w};
#pragma unroll
          for (int v = 0; v < 4; ++v) Bex[c][v] = p.j1 * ((xs[v] + zs[v]) + (own[c][v] + own[c][v + 2]));
        } else {
          // 4 in-plane nn (J1), 2 out-of-plane (J2), 4 in-plane nnn (J3): "4 nearest + 6 next nearest"
          float xs[6];
          xs[0] = lds1(next + left_b + cl) + lds1(prev + left_b + cl);
          xs[1] = xp.x + xm.x; xs[2] = xp.y + xm.y; xs[3] = xp.z + xm.z; xs[4] = xp.w + xm.w;
          xs[5] = lds1(next + right_b + cr) + lds1(prev + right_b + cr);
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            const float s1 = xs[v + 1] + (own[c][v] + own[c][v + 2]);
            const float s3 = xs[v] + xs[v + 2];
            Bex[c][v] = fmaf(p.j3, s3, fmaf(p.j2, zs[v], p.j1 * s1));
          }
        }
      }
      const uint32_t an = anbox + (uint32_t)(n & 1) * p.an_pitch + (uint32_t)(16 * g);
      const float4 ax4 = lds4(an), ay4 = lds4(an + row_b), az4 = lds4(an + 2u * row_b), ak4 = lds4(an + 3u * row_b);
      const float ax[4] = {ax4.x, ax4.y, ax4.z, ax4.w}, ay[4] = {ay4.x, ay4.y, ay4.z, ay4.w},
                  az[4] = {az4.x, az4.y, az4.z, az4.w}, ak[4] = {ak4.x, ak4.y, ak4.z, ak4.w};

      const float sg[4] = {sg4.x, sg4.y, sg4.z, sg4.w};
      const float bx[4] = {bx4.x, bx4.y, bx4.z, bx4.w}, by[4] = {by4.x, by4.y, by4.z, by4.w},
                  bz[4] = {bz4.x, bz4.y, bz4.z, bz4.w};
      float Ain[3][4];
      if (STAGE == 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { Ain[c][0] = a4[c].x; Ain[c][1] = a4[c].y; Ain[c][2] = a4[c].z; Ain[c][3] = a4[c].w; }
      }
      // ---- noise (in registers), torque, update, renormalise ----
      float o[3][4], oA[3][4];
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        uint32_t rnd[4];
        philox_site(p.key, n_lo, n_hi, gsite + (uint64_t)v, 0u, rnd);
        float xi[3];
        normals3(rnd, xi);
        const float Xs[3] = {own[0][v + 1], own[1][v + 1], own[2][v + 1]};
        const float Be[3] = {Bex[0][v], Bex[1][v], Bex[2][v]};
        const float Bap[3] = {bx[v], by[v], bz[v]};
        const float Ai[3] = {Ain[0][v], Ain[1][v], Ain[2][v]};
        float ov[3], oAv[3];
        site_update<STAGE>(sc, Xs, Be, make_float4(ax[v], ay[v], az[v], ak[v]), Bap, sg[v], xi, Ai, ov, oAv);
        o[0][v] = ov[0]; o[1][v] = ov[1]; o[2][v] = ov[2];
        if (STAGE == 0) { oA[0][v] = oAv[0]; oA[1][v] = oAv[1]; oA[2][v] = oAv[2]; }
      }
#pragma unroll
      for (int c = 0; c < 3; ++c)
        *reinterpret_cast<float4*>(p.arrays_w + (p.oOut + (uint32_t)c * p.as + e)) =
            make_float4(o[c][0], o[c][1], o[c][2], o[c][3]);
      if (STAGE == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c)
          *reinterpret_cast<float4*>(p.arrays_w + (p.oOutA + (uint32_t)c * p.as + e)) =
              make_float4(oA[c][0], oA[c][1], oA[c][2], oA[c][3]);
      }
    }
    e += planep;
    gsite += gplane;
    // this warp is done with slot n % kSlots (plane i-1) and with anisotropy box n & 1
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(bar_empty + 8u * (uint32_t)(n & (kSlots - 1)));
    if (tid == 0 && n + kSlots <= L + 1) {
      mbar_wait(bar_empty + 8u * (uint32_t)(n & (kSlots - 1)), (uint32_t)(n >> 2) & 1u);   // ... and so is every warp
      issue(n + kSlots);
    }
  }
}

// ---- host side ----
typedef void (*StageKernel)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const TmaParams);

// Compiled CTA shapes (threads, minimum CTAs per SM -> register budget): 384 x 2 -> 80, 320 x 2 -> 96, 256 x 3 -> 80.
struct Shape { int nt, minb; };
constexpr Shape kShapes[] = {{256, 3}, {320, 2}, {384, 2}};
constexpr int kNumShapes = 3;

template <int LAT, int STAGE>
StageKernel kernel_for(int shape) {
  switch (shape) {
    case 0: return heun_stage_tma<LAT, STAGE, 256, 3>;
    case 1: return heun_stage_tma<LAT, STAGE, 320, 2>;
    default: return heun_stage_tma<LAT, STAGE, 384, 2>;
  }
}
StageKernel kernel_for(int lattice, int stage, int shape) {
  if (lattice == ASD_SC) return stage == 0 ? kernel_for<LAT_SC, 0>(shape) : kernel_for<LAT_SC, 1>(shape);
  return stage == 0 ? kernel_for<LAT_L10, 0>(shape) : kernel_for<LAT_L10, 1>(shape);
}

}  // namespace

struct TmaPlan {
  CUtensorMap mapMain, mapEdge, mapAn;
  StageKernel kern[2] = {nullptr, nullptr};
  int32_t BY = 0, G = 0, nstrips = 0, CX = 0, nchunks = 0, threads = 0, ctas_per_sm = 0;
  uint32_t main_pitch = 0, edge_pitch = 0, an_pitch = 0, smem_bytes = 0;
};

// Same lattices as the film kernel, plus: a strip plan whose ring fits in shared memory.
bool heun_tma_supported(const Ctx& c) { return heun_fast_supported(c) && c.d.nz + 2 <= 256; }

namespace {

struct Candidate { int by, shape, ctas; double score; uint32_t smem; };

// Shared-memory bytes of a plan with strip width by.
uint32_t plan_smem(int nz, int by, uint32_t& main_pitch, uint32_t& edge_pitch, uint32_t& an_pitch) {
  main_pitch = (uint32_t)align_up((size_t)3 * (nz + 2) * by * 4, 128);
  edge_pitch = (uint32_t)align_up((size_t)3 * (nz + 2) * 16, 128);
  an_pitch = (uint32_t)align_up((size_t)16 * by, 128);
  return 128u + kSlots * (main_pitch + 2u * edge_pitch) + 2u * an_pitch;
}

// Builds (once per context) the strip / chunk plan and the tensor maps.
bool build_plan(Ctx& c, TmaPlan& pl) {
  if (!heun_tma_supported(c)) return false;
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const int ny = c.d.ny, nz = c.d.nz, nx = c.d.nx;
  int smem_sm = 0, smem_cta = 0;
  cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, c.device);
  cudaDeviceGetAttribute(&smem_cta, cudaDevAttrMaxSharedMemoryPerBlockOptin, c.device);

  // Strip width: every multiple of 4 up to 64 sites is tried; a plan is scored by the fraction of lanes that own
  // real sites (ragged last strip, ragged last warp) times a mild preference for >= 20 resident warps per SM and for
  // the spill-free CTA shape.
  const char* force = std::getenv("ASD_TMA_BY");          // tuning override (strip width in sites)
  const int force_by = force ? std::atoi(force) : 0;
  Candidate best{0, 0, 0, -1.0, 0};
  for (int by = 4; by <= 64; by += 4) {
    if (force_by && by != force_by) continue;
    const int ns = (ny + by - 1) / by, tasks = nz * (by / 4);
    uint32_t mp, ep, ap;
    const uint32_t smem = plan_smem(nz, by, mp, ep, ap);
    if ((int)smem > smem_cta) continue;
    for (int sh = 0; sh < kNumShapes; ++sh) {
      if (tasks > kShapes[sh].nt) continue;
      int ctas = smem_sm / (int)(smem + 1024);
      if (ctas > kShapes[sh].minb) ctas = kShapes[sh].minb;
      if (ctas < 1) continue;
      const double lanes = ((double)ny / (ns * by)) * ((double)tasks / kShapes[sh].nt);
      const double warps = ctas * kShapes[sh].nt / 32.0;
      // the 96-register shape (320 x 2) has no spills: measured 66 us per cfg4 stage against 76 us for 384 x 2
      const double score = lanes * (warps >= 20.0 ? 1.0 : warps / 20.0) * (kShapes[sh].nt == 320 ? 1.15 : 1.0);
      if (score > best.score) best = Candidate{by, sh, ctas, score, smem};
      break;                                                // smallest shape that holds the tasks
    }
  }
  if (best.score < 0.0) return false;
  pl.BY = best.by; pl.G = best.by / 4; pl.nstrips = (ny + best.by - 1) / best.by;
  pl.threads = kShapes[best.shape].nt;
  pl.smem_bytes = plan_smem(nz, pl.BY, pl.main_pitch, pl.edge_pitch, pl.an_pitch);
  int bps_min = 1 << 30;
  for (int st = 0; st < 2; ++st) {
    pl.kern[st] = kernel_for(c.d.lattice, st, best.shape);
    int bps = 0;
    if (cudaFuncSetAttribute((const void*)pl.kern[st], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, (const void*)pl.kern[st], pl.threads, pl.smem_bytes) != cudaSuccess ||
        bps < 1) {
      cudaGetLastError();
      return false;
    }
    if (bps < bps_min) bps_min = bps;
  }
  pl.ctas_per_sm = bps_min;
  // one wave: as many x-chunks as there are CTA slots for each strip
  int nchunks = (c.sm_count * bps_min) / pl.nstrips;
  if (nchunks < 1) nchunks = 1;
  if (nchunks > nx) nchunks = nx;
  pl.CX = (nx + nchunks - 1) / nchunks;
  pl.nchunks = (nx + pl.CX - 1) / pl.CX;

  // The 13 per-site arrays as one 4-D tensor (y, z-row, x-plane, array); origin = site (0,0,0) of array 0.
  const cuuint64_t dims[4] = {(cuuint64_t)ny, (cuuint64_t)nz, (cuuint64_t)nx, (cuuint64_t)AR_COUNT};
  const cuuint64_t strides[3] = {(cuuint64_t)c.nyp * 4, (cuuint64_t)nz * c.nyp * 4, (cuuint64_t)c.as * 4};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const cuuint32_t box_main[4] = {(cuuint32_t)pl.BY, (cuuint32_t)(nz + 2), 1u, 3u};
  const cuuint32_t box_edge[4] = {4u, (cuuint32_t)(nz + 2), 1u, 3u};
  if (enc(&pl.mapMain, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)(c.arrays + c.lead), dims, strides, box_main, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return false;
  if (enc(&pl.mapEdge, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)(c.arrays + c.lead), dims, strides, box_edge, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return false;
  // anisotropy table: (y, track plane, component)
  {
    const cuuint64_t ncol = (cuuint64_t)c.d.track_nx * (cuuint64_t)ny;
    const cuuint64_t adims[3] = {(cuuint64_t)ny, (cuuint64_t)c.d.track_nx, 4};
    const cuuint64_t astrides[2] = {(cuuint64_t)ny * 4, ncol * 4};
    const cuuint32_t abox[3] = {(cuuint32_t)pl.BY, 1u, 4u};
    if (enc(&pl.mapAn, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)c.aniso, adims, astrides, abox, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  return true;
}

}  // namespace

TmaPlan* tma_plan(Ctx& c) {
  if (!c.tma_plan_tried) {
    c.tma_plan_tried = true;
    TmaPlan* pl = new TmaPlan();
    if (build_plan(c, *pl)) c.tma_plan = pl;
    else delete pl;
  }
  return c.tma_plan;
}

void tma_plan_free(Ctx& c) {
  delete c.tma_plan;
  c.tma_plan = nullptr;
}

asd_status launch_heun_tma(Ctx& c, StageParams& p) {
  TmaPlan* pl = tma_plan(c);
  if (!pl) return ASD_EUNSUPPORTED;
  TmaParams f;
  f.arrays = c.arrays; f.arrays_w = c.arrays; f.as = (uint32_t)c.as;
  f.oSigma = AR_SIGMA * f.as; f.oB = AR_B * f.as;
  f.nx = c.d.nx; f.ny = c.d.ny; f.nz = c.d.nz; f.nyp = c.nyp; f.lead = c.lead;
  f.BY = pl->BY; f.G = pl->G; f.nstrips = pl->nstrips; f.CX = pl->CX;
  f.x0 = (int32_t)c.x0;
  f.main_pitch = pl->main_pitch; f.edge_pitch = pl->edge_pitch; f.an_pitch = pl->an_pitch;
  f.j1 = p.jx[0]; f.j2 = p.jx[1]; f.j3 = p.jx[2];
  f.gdt = p.gdt; f.lambda = p.lambda; f.scale = p.scale;
  f.n_lo = p.n_lo; f.n_hi = p.n_hi; f.dyn = p.dyn; f.g0 = p.g0; f.key = p.key;
  const unsigned blocks = (unsigned)(pl->nstrips * pl->nchunks);
  const uint32_t as = f.as;
  // predictor: X = S -> S~, A
  f.aX = c.aS; f.oOut = (uint32_t)c.aSt * as; f.oOutA = AR_A * as; f.oA = AR_A * as;
  pl->kern[0]<<<blocks, pl->threads, pl->smem_bytes, c.launch_stream>>>(pl->mapMain, pl->mapEdge, pl->mapAn, f);
  ASD_LAUNCH_CHECK(c, "heun predictor (tma)");
  // corrector: X = S~, A -> S
  f.aX = c.aSt; f.oOut = (uint32_t)c.aS * as;
  pl->kern[1]<<<blocks, pl->threads, pl->smem_bytes, c.launch_stream>>>(pl->mapMain, pl->mapEdge, pl->mapAn, f);
  ASD_LAUNCH_CHECK(c, "heun corrector (tma)");
  return ASD_OK;
}

}  // namespace asd
