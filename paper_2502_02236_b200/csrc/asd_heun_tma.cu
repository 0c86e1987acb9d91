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

#include "asd_internal.cuh"
#include "asd_site.cuh"

namespace asd {

namespace {

constexpr int LAT_SC = 0, LAT_L10 = 1;
constexpr int kSlots = 4;          // ring of X planes: i-1, i, i+1 in use, i+2 in flight
constexpr int kYLead = 4;          // the box starts 4 sites before the strip: own sites sit 16-byte aligned
constexpr int kMaxThreads = 384;

struct TmaParams {
  const float* arrays;
  float* arrays_w;
  uint32_t as;                     // array stride (elements)
  int32_t aX;                      // array index of component 0 of the configuration read through the TMA
  uint32_t oA, oOut, oOutA, oSigma, oB;   // element offsets (array index * as)
  int32_t nx, ny, nz, nyp, lead;
  int32_t BY, G, nstrips, CX;      // strip width (sites), y-groups per strip row (BY / 4), strips, planes per chunk
  int32_t x0;                      // global plane of window plane 0 (anisotropy table coordinate)
  uint32_t slot_bytes, an_bytes;   // shared-memory pitch of one X-plane box / one anisotropy box (multiples of 128)
  uint32_t x_bytes;                // exact bytes of one X-plane box (what the TMA reports to the mbarrier)
  float j1, j2, j3;
  float gdt, lambda, scale;
  uint32_t n_lo, n_hi;
  uint64_t g0;
  PhiloxKey key;
};

// ---- PTX wrappers: mbarrier and bulk tensor copies ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0u;
}
// try_wait suspends the thread in hardware for a bounded time per attempt; a transaction count that can never
// complete (a programming error) traps after ~2^24 attempts instead of hanging the device.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t spins = 0;
  while (!mbar_try_wait(bar, parity)) {
    if (++spins > (1u << 24)) __trap();
  }
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2,
                                            int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ float4 ldg_stream4(const float* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ float4 lds4(const float* p) { return *reinterpret_cast<const float4*>(p); }

// Shared memory: [kSlots mbarriers, padded to 128 B][kSlots X-plane boxes][2 anisotropy boxes].
// X-plane box (one TMA): float [3 components][nz + 2 rows (z = -1 .. nz)][BYH = BY + 8 sites (y = j0-4 .. j0+BY+3)].
// Anisotropy box: float [4][BY].
template <int LAT, int STAGE>
__global__ void __launch_bounds__(kMaxThreads, 2)
heun_stage_tma(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapAn, const TmaParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const uint32_t bar0 = smem_u32(smem_raw);
  const float* slots = reinterpret_cast<const float*>(smem_raw + 128);
  const float* anbox = reinterpret_cast<const float*>(smem_raw + 128 + kSlots * p.slot_bytes);
  const uint32_t slot_f = p.slot_bytes >> 2, an_f = p.an_bytes >> 2;

  const int tid = (int)threadIdx.x;
  const int strip = (int)blockIdx.x % p.nstrips, chunk = (int)blockIdx.x / p.nstrips;
  const int j0 = strip * p.BY;
  const int i_begin = chunk * p.CX;
  const int L = min(p.CX, p.nx - i_begin);            // planes of this CTA
  const int BYH = p.BY + 2 * kYLead;

  // plane m of the march (m = 0 is window plane i_begin - 1, the trailing halo) -> slot m & 3; the anisotropy box of
  // march step n = m - 2 rides on the same barrier.
  auto issue = [&](int m) {
    const uint32_t bar = bar0 + 8u * (uint32_t)(m & (kSlots - 1));
    const int n = m - 2;
    const bool with_an = (n >= 0 && n < L);
    mbar_expect_tx(bar, p.x_bytes + (with_an ? (uint32_t)(4 * p.BY * 4) : 0u));
    tma_load_4d(smem_u32(slots) + (uint32_t)(m & (kSlots - 1)) * p.slot_bytes, &mapX, bar, j0 - kYLead, -1,
                i_begin - 1 + m, p.aX);
    if (with_an) tma_load_3d(smem_u32(anbox) + (uint32_t)(n & 1) * p.an_bytes, &mapAn, bar, j0, p.x0 + i_begin + n, 0);
  };

  if (tid == 0) {
    for (int s = 0; s < kSlots; ++s) mbar_init(bar0 + 8u * s, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (int m = 0; m < kSlots && m <= L + 1; ++m) issue(m);
  }
  __syncthreads();

  // ---- this thread's (row, y-group): fixed for the whole march ----
  const int k = tid / p.G, g = tid - k * p.G;
  const int j = j0 + 4 * g;
  const bool active = (k < p.nz) && (j < p.ny);
  // float index of the first own site inside a component of an X box: row k+1 (row 0 is z = -1), site kYLead + 4g
  const uint32_t own_f = (uint32_t)((k + 1) * BYH + kYLead + 4 * g);
  const uint32_t comp_f = (uint32_t)((p.nz + 2) * BYH);
  uint32_t e = (uint32_t)(p.lead + (i_begin * p.nz + k) * p.nyp + j);      // padded element of the first own site
  const uint32_t planep = (uint32_t)(p.nz * p.nyp);
  uint64_t gsite = p.g0 + (uint64_t)((uint32_t)(i_begin * p.nz + k) * (uint32_t)p.ny + (uint32_t)j);
  const uint32_t gplane = (uint32_t)(p.nz * p.ny);
  const SiteConst sc{p.gdt, p.lambda, p.scale};

  mbar_wait(bar0 + 0u, 0u);
  mbar_wait(bar0 + 8u, 0u);

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
      mbar_wait(bar0 + 8u * (uint32_t)(m & (kSlots - 1)), (uint32_t)(m >> 2) & 1u);
    }
    if (active) {
      const float* prev = slots + (uint32_t)(n & (kSlots - 1)) * slot_f + own_f;
      const float* cur = slots + (uint32_t)((n + 1) & (kSlots - 1)) * slot_f + own_f;
      const float* next = slots + (uint32_t)((n + 2) & (kSlots - 1)) * slot_f + own_f;

      // ---- exchange field, Eq. (2): shell sums first, one multiply per shell ----
      float own[3][6];                // own row with its y-1 and y+1 edge sites
      float Bex[3][4];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float* qc = cur + (uint32_t)c * comp_f;
        const float* qn = next + (uint32_t)c * comp_f;
        const float* qp = prev + (uint32_t)c * comp_f;
        const float4 o = lds4(qc);
        own[c][0] = qc[-1]; own[c][1] = o.x; own[c][2] = o.y; own[c][3] = o.z; own[c][4] = o.w; own[c][5] = qc[4];
        const float4 zp = lds4(qc + BYH), zm = lds4(qc - BYH);
        const float4 xp = lds4(qn), xm = lds4(qp);
        const float zs[4] = {zp.x + zm.x, zp.y + zm.y, zp.z + zm.z, zp.w + zm.w};
        if (LAT == LAT_SC) {
          // 6 nearest neighbours, one J
          const float xs[4] = {xp.x + xm.x, xp.y + xm.y, xp.z + xm.z, xp.w + xm.w};
#pragma unroll
          for (int v = 0; v < 4; ++v) Bex[c][v] = p.j1 * ((xs[v] + zs[v]) + (own[c][v] + own[c][v + 2]));
        } else {
          // 4 in-plane nn (J1), 2 out-of-plane (J2), 4 in-plane nnn (J3): "4 nearest + 6 next nearest"
          float xs[6];
          xs[0] = qn[-1] + qp[-1];
          xs[1] = xp.x + xm.x; xs[2] = xp.y + xm.y; xs[3] = xp.z + xm.z; xs[4] = xp.w + xm.w;
          xs[5] = qn[4] + qp[4];
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            const float s1 = xs[v + 1] + (own[c][v] + own[c][v + 2]);
            const float s3 = xs[v] + xs[v + 2];
            Bex[c][v] = fmaf(p.j3, s3, fmaf(p.j2, zs[v], p.j1 * s1));
          }
        }
      }
      const float* an = anbox + (uint32_t)(n & 1) * an_f + 4 * g;
      const float4 ax4 = lds4(an), ay4 = lds4(an + p.BY), az4 = lds4(an + 2 * p.BY), ak4 = lds4(an + 3 * p.BY);
      const float ax[4] = {ax4.x, ax4.y, ax4.z, ax4.w}, ay[4] = {ay4.x, ay4.y, ay4.z, ay4.w},
                  az[4] = {az4.x, az4.y, az4.z, az4.w}, ak[4] = {ak4.x, ak4.y, ak4.z, ak4.w};

      // ---- noise (in registers) ----
      float xi[4][3];
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        uint32_t rnd[4];
        philox_site(p.key, p.n_lo, p.n_hi, gsite + (uint64_t)v, 0u, rnd);
        normals3(rnd, xi[v]);
      }

      // ---- torque, update, renormalise ----
      const float sg[4] = {sg4.x, sg4.y, sg4.z, sg4.w};
      const float bx[4] = {bx4.x, bx4.y, bx4.z, bx4.w}, by[4] = {by4.x, by4.y, by4.z, by4.w},
                  bz[4] = {bz4.x, bz4.y, bz4.z, bz4.w};
      float Ain[3][4];
      if (STAGE == 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { Ain[c][0] = a4[c].x; Ain[c][1] = a4[c].y; Ain[c][2] = a4[c].z; Ain[c][3] = a4[c].w; }
      }
      float o[3][4], oA[3][4];
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float Xs[3] = {own[0][v + 1], own[1][v + 1], own[2][v + 1]};
        const float Be[3] = {Bex[0][v], Bex[1][v], Bex[2][v]};
        const float Bap[3] = {bx[v], by[v], bz[v]};
        const float Ai[3] = {Ain[0][v], Ain[1][v], Ain[2][v]};
        float ov[3], oAv[3];
        site_update<STAGE>(sc, Xs, Be, make_float4(ax[v], ay[v], az[v], ak[v]), Bap, sg[v], xi[v], Ai, ov, oAv);
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
    __syncthreads();                                         // every thread is done with slot n & 3 and anisotropy box n & 1
    if (tid == 0 && n + kSlots <= L + 1) issue(n + kSlots);
  }
}

// ---- host side ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)ptr;
  }
  return fn;
}

}  // namespace

struct TmaPlan {
  bool ok = false;
  CUtensorMap mapX, mapAn;
  int32_t BY = 0, G = 0, nstrips = 0, CX = 0, nchunks = 0, threads = 0;
  uint32_t slot_bytes = 0, an_bytes = 0, smem_bytes = 0;
};

namespace {

template <int LAT, int STAGE>
bool configure(uint32_t smem, int threads, int& blocks_per_sm) {
  if (cudaFuncSetAttribute(heun_stage_tma<LAT, STAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
      cudaSuccess)
    return false;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, heun_stage_tma<LAT, STAGE>, threads, smem) ==
             cudaSuccess && blocks_per_sm >= 1;
}

}  // namespace

// Same lattices as the film kernel, plus: a strip plan whose ring fits in shared memory.
bool heun_tma_supported(const Ctx& c) { return heun_fast_supported(c) && c.d.nz + 2 <= 256; }

// Builds (once per context) the tensor maps and the strip / chunk plan.
static bool build_plan(Ctx& c, TmaPlan& pl) {
  if (!heun_tma_supported(c)) return false;
  EncodeTiledFn enc = encode_fn();
  if (!enc) return false;
  const int ny = c.d.ny, nz = c.d.nz, nx = c.d.nx;
  // strip width: as few strips as keep a strip row <= byMax sites and the CTA <= kMaxThreads threads
  int best_by = 0;
  for (int by_max = 64; by_max >= 4 && !best_by; by_max -= 4) {
    const int ns = (ny + by_max - 1) / by_max;
    const int by = (int)align_up((size_t)((ny + ns - 1) / ns), 4);
    const int threads = (int)align_up((size_t)(nz * (by / 4)), 32);
    const size_t slot = align_up((size_t)3 * (nz + 2) * (by + 2 * kYLead) * 4, 128);
    const size_t smem = 128 + kSlots * slot + 2 * align_up((size_t)16 * by, 128);
    if (threads <= kMaxThreads && smem <= 110 * 1024) best_by = by;
  }
  if (!best_by) return false;
  pl.BY = best_by; pl.G = best_by / 4; pl.nstrips = (ny + best_by - 1) / best_by;
  pl.threads = (int)align_up((size_t)(nz * pl.G), 32);
  pl.slot_bytes = (uint32_t)align_up((size_t)3 * (nz + 2) * (pl.BY + 2 * kYLead) * 4, 128);
  pl.an_bytes = (uint32_t)align_up((size_t)16 * pl.BY, 128);
  pl.smem_bytes = 128 + kSlots * pl.slot_bytes + 2 * pl.an_bytes;

  int bps = 0, bps_min = 1 << 30;
  const bool sc = c.d.lattice == ASD_SC;
  bool okc = sc ? configure<LAT_SC, 0>(pl.smem_bytes, pl.threads, bps) : configure<LAT_L10, 0>(pl.smem_bytes, pl.threads, bps);
  if (!okc) { cudaGetLastError(); return false; }
  bps_min = bps;
  okc = sc ? configure<LAT_SC, 1>(pl.smem_bytes, pl.threads, bps) : configure<LAT_L10, 1>(pl.smem_bytes, pl.threads, bps);
  if (!okc) { cudaGetLastError(); return false; }
  if (bps < bps_min) bps_min = bps;
  // one wave: as many x-chunks as there are CTA slots for each strip
  const int slots = c.sm_count * bps_min;
  int nchunks = slots / pl.nstrips;
  if (nchunks < 1) nchunks = 1;
  if (nchunks > nx) nchunks = nx;
  pl.CX = (nx + nchunks - 1) / nchunks;
  pl.nchunks = (nx + pl.CX - 1) / pl.CX;

  // X: the 13 per-site arrays as one 4-D tensor (y, z-row, x-plane, array); origin = site (0,0,0) of array 0
  {
    const cuuint64_t dims[4] = {(cuuint64_t)ny, (cuuint64_t)nz, (cuuint64_t)nx, (cuuint64_t)AR_COUNT};
    const cuuint64_t strides[3] = {(cuuint64_t)c.nyp * 4, (cuuint64_t)nz * c.nyp * 4, (cuuint64_t)c.as * 4};
    const cuuint32_t box[4] = {(cuuint32_t)(pl.BY + 2 * kYLead), (cuuint32_t)(nz + 2), 1u, 3u};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    if (enc(&pl.mapX, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)(c.arrays + c.lead), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  // anisotropy table: (y, track plane, component)
  {
    const cuuint64_t ncol = (cuuint64_t)c.d.track_nx * (cuuint64_t)ny;
    const cuuint64_t dims[3] = {(cuuint64_t)ny, (cuuint64_t)c.d.track_nx, 4};
    const cuuint64_t strides[2] = {(cuuint64_t)ny * 4, ncol * 4};
    const cuuint32_t box[3] = {(cuuint32_t)pl.BY, 1u, 4u};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (enc(&pl.mapAn, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)c.aniso, dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  pl.ok = true;
  return true;
}

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

namespace {

template <int LAT>
asd_status launch_pair_tma(Ctx& c, const TmaPlan& pl, TmaParams& f) {
  const unsigned blocks = (unsigned)(pl.nstrips * pl.nchunks);
  const uint32_t as = f.as;
  f.aX = c.aS; f.oOut = (uint32_t)c.aSt * as; f.oOutA = AR_A * as; f.oA = AR_A * as;
  heun_stage_tma<LAT, 0><<<blocks, pl.threads, pl.smem_bytes, c.stream>>>(pl.mapX, pl.mapAn, f);
  ASD_LAUNCH_CHECK(c, "heun predictor (tma)");
  f.aX = c.aSt; f.oOut = (uint32_t)c.aS * as;
  heun_stage_tma<LAT, 1><<<blocks, pl.threads, pl.smem_bytes, c.stream>>>(pl.mapX, pl.mapAn, f);
  ASD_LAUNCH_CHECK(c, "heun corrector (tma)");
  return ASD_OK;
}

}  // namespace

asd_status launch_heun_tma(Ctx& c, StageParams& p) {
  TmaPlan* pl = tma_plan(c);
  if (!pl) return ASD_EUNSUPPORTED;
  TmaParams f;
  f.arrays = c.arrays; f.arrays_w = c.arrays; f.as = (uint32_t)c.as;
  f.oSigma = AR_SIGMA * f.as; f.oB = AR_B * f.as;
  f.nx = c.d.nx; f.ny = c.d.ny; f.nz = c.d.nz; f.nyp = c.nyp; f.lead = c.lead;
  f.BY = pl->BY; f.G = pl->G; f.nstrips = pl->nstrips; f.CX = pl->CX;
  f.x0 = (int32_t)c.x0;
  f.slot_bytes = pl->slot_bytes; f.an_bytes = pl->an_bytes;
  f.x_bytes = (uint32_t)(3 * (c.d.nz + 2) * (pl->BY + 2 * kYLead) * 4);
  f.j1 = p.jx[0]; f.j2 = p.jx[1]; f.j3 = p.jx[2];
  f.gdt = p.gdt; f.lambda = p.lambda; f.scale = p.scale;
  f.n_lo = p.n_lo; f.n_hi = p.n_hi; f.g0 = p.g0; f.key = p.key;
  return c.d.lattice == ASD_SC ? launch_pair_tma<LAT_SC>(c, *pl, f) : launch_pair_tma<LAT_L10>(c, *pl, f);
}

}  // namespace asd
