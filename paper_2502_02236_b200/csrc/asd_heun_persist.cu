// asd_heun_persist.cu -- the hot path for lattices that fit on chip (BASELINE configs[0]: 16^3 periodic): n stochastic
// Heun steps in ONE launch by ONE thread-block cluster, the lattice resident in shared memory for the whole call.
//
// A 4096-site lattice finishes a stage kernel in ~2 us, less than it costs to launch it ("cfg 0 is
// launch/latency-bound ... one persistent CTA"); graphs and dependent launches bring a Heun step to 8 us.  Here the
// window is cut along x into as many slabs as the cluster has CTAs (16 where the device schedules it, else 8, the
// portable maximum); every CTA keeps its slab of
// S and S~ in its own shared memory, one thread owning VEC (1, 2 or 4) consecutive y-sites with A = S + dt/2 k1, the
// noise xi and the site's constants in registers (VEC is chosen so that a CTA has as many warps as fit: a slab of a few
// hundred sites is latency-bound, and warps are what hides latency).  The x+-1 planes of a slab's first / last plane live in
// the neighbouring CTA's shared memory and are read there directly (distributed shared memory), so nothing but the final
// spins ever goes back to HBM.  Two cluster barriers per Heun step (S~ complete; S complete).
//
// Same arithmetic as the stage kernels (asd_site.cuh, asd_rng.cuh): Philox keyed by (seed; step, global site), the same
// xi in both stages.  Periodic wraps and open edges by index arithmetic; vacant sites hold 0, so a vacant neighbour drops
// out of Eq. (2) by itself -- which needs grains that do not touch (or one grain), checked by the dispatcher.
#include <cooperative_groups.h>
#include <cstdlib>

#include "asd_internal.cuh"
#include "asd_site.cuh"

namespace cg = cooperative_groups;

namespace asd {

namespace {

constexpr int LAT_SC = 0, LAT_L10 = 1;

struct PersistParams {
  float* arrays;
  uint32_t as;
  uint32_t oS, oSigma, oB;          // element offsets of S component 0, sigma, B component 0
  const uint32_t* col;
  const float4* grain;
  int32_t nx, ny, nz, nyp, lead;
  int32_t ppc;                      // planes per CTA
  int32_t pbc_x, pbc_y, pbc_z;
  float j1, j2, j3, gdt, lambda, scale;
  uint64_t step0;                   // index of the first step
  int32_t nsteps;
  uint64_t g0;
  PhiloxKey key;
};

template <int VEC> struct PV;
template <> struct PV<1> {
  static __device__ __forceinline__ void ld(const float* p, float v[1]) { v[0] = *p; }
  static __device__ __forceinline__ void st(float* p, const float v[1]) { *p = v[0]; }
};
template <> struct PV<2> {
  static __device__ __forceinline__ void ld(const float* p, float v[2]) { const float2 t = *reinterpret_cast<const float2*>(p); v[0] = t.x; v[1] = t.y; }
  static __device__ __forceinline__ void st(float* p, const float v[2]) { *reinterpret_cast<float2*>(p) = make_float2(v[0], v[1]); }
};
template <> struct PV<4> {
  static __device__ __forceinline__ void ld(const float* p, float v[4]) { const float4 t = *reinterpret_cast<const float4*>(p); v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w; }
  static __device__ __forceinline__ void st(float* p, const float v[4]) { *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]); }
};

// NT bounds the registers per thread (65536 / NT): every instance below keeps A, xi and the site constants of its VEC
// sites in registers except <4, 1024> (64 registers: the fallback for slabs of up to 4096 sites per CTA; it spills).
template <int LAT, int VEC, int NT>
__global__ void __launch_bounds__(NT, 1) heun_persistent(const PersistParams p) {
  extern __shared__ __align__(16) float smem[];
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank(), ncta = (int)cluster.num_blocks();
  const int ny = p.ny, nz = p.nz, ppc = p.ppc;
  const int slab = ppc * nz * ny;
  const int ngrp = ny / VEC;
  const int t = (int)threadIdx.x;
  const bool active = t < ppc * nz * ngrp;
  const int r = active ? t / ngrp : 0;
  const int j0 = active ? (t - r * ngrp) * VEC : 0;
  const int li = r / nz, k = r - li * nz;
  const int i = rank * ppc + li;                                   // window plane
  const int own = r * ny + j0;                                     // own sites inside a component
  // neighbour CTAs' shared memory (generic pointers into distributed shared memory)
  const int rank_m = (rank == 0) ? ncta - 1 : rank - 1, rank_p = (rank == ncta - 1) ? 0 : rank + 1;
  const float* sm_m = cluster.map_shared_rank(smem, rank_m);
  const float* sm_p = cluster.map_shared_rank(smem, rank_p);
  // x-1 / x+1 rows: local plane, or the facing plane of the neighbouring slab; missing at an open window edge
  const bool xm_ok = (i > 0) || p.pbc_x, xp_ok = (i < p.nx - 1) || p.pbc_x;
  const float* xm_base = (li > 0) ? smem : sm_m;
  const float* xp_base = (li < ppc - 1) ? smem : sm_p;
  const int xm_row = ((li > 0 ? li - 1 : ppc - 1) * nz + k) * ny;
  const int xp_row = ((li < ppc - 1 ? li + 1 : 0) * nz + k) * ny;
  const bool zm_ok = (k > 0) || p.pbc_z, zp_ok = (k < nz - 1) || p.pbc_z;
  const int zm_row = (li * nz + (k > 0 ? k - 1 : nz - 1)) * ny;
  const int zp_row = (li * nz + (k < nz - 1 ? k + 1 : 0)) * ny;
  const int own_row = r * ny;
  // y-1 / y+VEC columns (wrap folded in); absent: open edge
  const bool yl_ok = (j0 > 0) || p.pbc_y, yr_ok = (j0 + VEC < ny) || p.pbc_y;
  const int jl = (j0 > 0) ? j0 - 1 : ny - 1, jr = (j0 + VEC < ny) ? j0 + VEC : 0;

  // ---- load: spins into shared memory, per-site constants into registers ----
  const uint32_t e = (uint32_t)(p.lead + (i * nz + k) * p.nyp + j0);
  float sg[VEC], Bap[3][VEC];
  float4 gp4[VEC];
#pragma unroll
  for (int v = 0; v < VEC; ++v) {
    sg[v] = 0.f; Bap[0][v] = Bap[1][v] = Bap[2][v] = 0.f;
    gp4[v] = make_float4(0.f, 0.f, 1.f, 0.f);
  }
  if (active) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      float sv[VEC];
      PV<VEC>::ld(p.arrays + (p.oS + (uint32_t)c * p.as + e), sv);
      PV<VEC>::st(smem + c * slab + own, sv);
      PV<VEC>::ld(p.arrays + (p.oB + (uint32_t)c * p.as + e), Bap[c]);
    }
    PV<VEC>::ld(p.arrays + (p.oSigma + e), sg);
#pragma unroll
    for (int v = 0; v < VEC; ++v)
      gp4[v] = __ldg(p.grain + (p.col[(uint32_t)i * (uint32_t)ny + (uint32_t)(j0 + v)] & 0xFFFFu));
  }
  cluster.sync();

  const SiteConst sc{p.gdt, p.lambda, p.scale};
  const uint64_t gsite = p.g0 + (uint64_t)((i * nz + k) * ny + j0);
  const float zero3[3] = {0.f, 0.f, 0.f};

  // Exchange field of the VEC own sites in configuration `cfg` (float offset of its component 0 inside a CTA's memory)
  auto exchange = [&](int cfg, float X[3][VEC], float Bex[3][VEC]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int cb = cfg + c * slab;
      const float* rowp = smem + cb + own_row;
      float ownv[VEC + 2];
      PV<VEC>::ld(rowp + j0, ownv + 1);
      ownv[0] = yl_ok ? rowp[jl] : 0.f; ownv[VEC + 1] = yr_ok ? rowp[jr] : 0.f;
      float zp[VEC], zm[VEC], xp[VEC + 2], xm[VEC + 2];
#pragma unroll
      for (int v = 0; v < VEC; ++v) { X[c][v] = ownv[v + 1]; zp[v] = 0.f; zm[v] = 0.f; }
#pragma unroll
      for (int v = 0; v < VEC + 2; ++v) { xp[v] = 0.f; xm[v] = 0.f; }
      if (zp_ok) PV<VEC>::ld(smem + cb + zp_row + j0, zp);
      if (zm_ok) PV<VEC>::ld(smem + cb + zm_row + j0, zm);
      const float* xpr = xp_base + cb + xp_row;
      const float* xmr = xm_base + cb + xm_row;
      if (xp_ok) PV<VEC>::ld(xpr + j0, xp + 1);
      if (xm_ok) PV<VEC>::ld(xmr + j0, xm + 1);
      if (LAT == LAT_SC) {
        // 6 nearest neighbours, one J
#pragma unroll
        for (int v = 0; v < VEC; ++v)
          Bex[c][v] = p.j1 * (((xp[v + 1] + xm[v + 1]) + (zp[v] + zm[v])) + (ownv[v] + ownv[v + 2]));
      } else {
        // 4 in-plane nn (J1), 2 out-of-plane (J2), 4 in-plane nnn (J3): "4 nearest + 6 next nearest"
        if (xp_ok && yl_ok) xp[0] = xpr[jl];
        if (xp_ok && yr_ok) xp[VEC + 1] = xpr[jr];
        if (xm_ok && yl_ok) xm[0] = xmr[jl];
        if (xm_ok && yr_ok) xm[VEC + 1] = xmr[jr];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
          const float s1 = (xp[v + 1] + xm[v + 1]) + (ownv[v] + ownv[v + 2]);
          const float s3 = (xp[v] + xm[v]) + (xp[v + 2] + xm[v + 2]);
          Bex[c][v] = fmaf(p.j3, s3, fmaf(p.j2, zp[v] + zm[v], p.j1 * s1));
        }
      }
    }
  };

  // The noise of a step depends on nothing but its counters: it is drawn between the ARRIVAL at the barrier that closes
  // the previous step and the WAIT for it, so that the barrier's latency hides behind Philox and Box-Muller.
  float xi[VEC][3];
  auto draw = [&](uint64_t n) {
    const uint32_t n_lo = (uint32_t)n, n_hi = (uint32_t)(n >> 32);
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
      uint32_t rnd[4];
      philox_site(p.key, n_lo, n_hi, gsite + (uint64_t)v, 0u, rnd);
      normals3(rnd, xi[v]);
    }
  };
  draw(p.step0);
  for (int s = 0; s < p.nsteps; ++s) {
    float A[3][VEC];
    // ---- predictor: S~ = normalise(S + dt k1), A = S + dt/2 k1 ----
    if (active) {
      float X[3][VEC], Bex[3][VEC];
      exchange(0, X, Bex);
#pragma unroll
      for (int v = 0; v < VEC; ++v) {
        const float Xs[3] = {X[0][v], X[1][v], X[2][v]};
        const float Be[3] = {Bex[0][v], Bex[1][v], Bex[2][v]};
        const float Ba[3] = {Bap[0][v], Bap[1][v], Bap[2][v]};
        float ov[3], oA[3];
        site_update<0>(sc, Xs, Be, gp4[v], Ba, sg[v], xi[v], zero3, ov, oA);
        A[0][v] = oA[0]; A[1][v] = oA[1]; A[2][v] = oA[2];
        X[0][v] = ov[0]; X[1][v] = ov[1]; X[2][v] = ov[2];
      }
#pragma unroll
      for (int c = 0; c < 3; ++c) PV<VEC>::st(smem + (3 + c) * slab + own, X[c]);
    }
    cluster.sync();                                  // S~ complete everywhere; nobody reads S any more
    // ---- corrector: S = normalise(A + dt/2 k2), same xi ----
    if (active) {
      float X[3][VEC], Bex[3][VEC];
      exchange(3 * slab, X, Bex);
#pragma unroll
      for (int v = 0; v < VEC; ++v) {
        const float Xs[3] = {X[0][v], X[1][v], X[2][v]};
        const float Be[3] = {Bex[0][v], Bex[1][v], Bex[2][v]};
        const float Ba[3] = {Bap[0][v], Bap[1][v], Bap[2][v]};
        const float Ai[3] = {A[0][v], A[1][v], A[2][v]};
        float ov[3], oA[3];
        site_update<1>(sc, Xs, Be, gp4[v], Ba, sg[v], xi[v], Ai, ov, oA);
        X[0][v] = ov[0]; X[1][v] = ov[1]; X[2][v] = ov[2];
      }
#pragma unroll
      for (int c = 0; c < 3; ++c) PV<VEC>::st(smem + c * slab + own, X[c]);
    }
    cluster.barrier_arrive();                        // this CTA's share of S is written ...
    if (s + 1 < p.nsteps) draw(p.step0 + (uint64_t)(s + 1));
    cluster.barrier_wait();                          // ... S complete everywhere; nobody reads S~ any more
  }

  if (active) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      float sv[VEC];
      PV<VEC>::ld(smem + c * slab + own, sv);
      PV<VEC>::st(p.arrays + (p.oS + (uint32_t)c * p.as + e), sv);
    }
  }
}

typedef void (*PersistKernel)(const PersistParams);
struct PersistShape { int ncta, ppc, vec, threads; size_t smem; PersistKernel kern; };

template <int LAT>
PersistKernel persist_kernel(int vec, int threads) {
  if (vec == 1) return heun_persistent<LAT, 1, 512>;
  if (vec == 2) return heun_persistent<LAT, 2, 512>;
  return threads <= 256 ? heun_persistent<LAT, 4, 256> : (threads <= 512 ? heun_persistent<LAT, 4, 512> : heun_persistent<LAT, 4, 1024>);
}

// Largest cluster (8, 4, 2, 1 CTAs) whose slabs are whole planes and fit a CTA's shared memory; then as few sites per
// thread as fit 512 threads (a slab this small is latency-bound: more warps hide more of it), else 4 per thread.
bool persist_shape(const Ctx& c, PersistShape& sh) {
  if (c.d.ny % 4 != 0) return false;
  int smem_cta = 0;
  cudaDeviceGetAttribute(&smem_cta, cudaDevAttrMaxSharedMemoryPerBlockOptin, c.device);
  // 16 CTAs per cluster is beyond the portable size: taken when the device can schedule it (asked once per shape below)
  int max_ncta = 16;                                      // measured on cfg0: 16 CTAs 1.32 us per Heun step, 8: 1.46, 4: 2.27
  if (const char* ev = std::getenv("ASD_PERSIST_CLUSTER")) max_ncta = std::atoi(ev);       // tuning override: 1, 2, 4, 8, 16
  for (int ncta = max_ncta; ncta >= 1; ncta >>= 1) {
    if (c.d.nx % ncta != 0) continue;
    const int ppc = c.d.nx / ncta;
    const int64_t sites = (int64_t)ppc * c.d.nz * c.d.ny;
    const size_t smem = sizeof(float) * 6 * (size_t)sites;
    if (sites / 4 > 1024 || smem > (size_t)smem_cta) continue;
    const int vec = sites <= 512 ? 1 : (sites / 2 <= 512 ? 2 : 4);
    sh.ncta = ncta; sh.ppc = ppc; sh.vec = vec; sh.threads = (int)((sites / vec + 31) / 32 * 32); sh.smem = smem;
    sh.kern = c.d.lattice == ASD_SC ? persist_kernel<LAT_SC>(vec, sh.threads) : persist_kernel<LAT_L10>(vec, sh.threads);
    if (ncta > 8) {                                       // non-portable cluster size: opt in, and ask whether it can run
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)ncta); cfg.blockDim = dim3((unsigned)sh.threads); cfg.dynamicSmemBytes = smem;
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeClusterDimension;
      attr[0].val.clusterDim.x = (unsigned)ncta; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
      cfg.attrs = attr; cfg.numAttrs = 1;
      int nclusters = 0;
      if (cudaFuncSetAttribute((const void*)sh.kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess ||
          cudaFuncSetAttribute((const void*)sh.kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
          cudaOccupancyMaxActiveClusters(&nclusters, (const void*)sh.kern, &cfg) != cudaSuccess || nclusters < 1) {
        cudaGetLastError();
        continue;
      }
    }
    return true;
  }
  return false;
}

}  // namespace

// Built-in shells, one grain or grains that do not touch (a vacant neighbour is a stored zero), 128-bit rows, no
// per-stage global quantity (demagnetising field, mesh coupling), and a lattice that fits one cluster.
bool heun_persist_supported(const Ctx& c) {
  PersistShape sh;
  return c.d.ell_width == 0 && !c.grains_touch && !c.demag && !edge_field_on(c) && (int64_t)AR_COUNT * c.as < (1ll << 31) &&
         persist_shape(c, sh);
}

// What ASD_KERNEL_AUTO asks: is the persistent cluster the fastest path for this lattice?  Measured on B200, us per Heun step,
// persistent against CUDA-graph replay of the stage kernels (film kernel 4.9-5.6, general kernel 8.0-9.4 whatever the size
// below 2^16 sites): simple cubic 1024 / 1536 / 2048 / 3072 sites per CTA: 2.3 / 3.5 / 3.7 / 8.1; L1_0 1024 / 1536 / 2048 /
// 3072: 3.3 / 6.2 / 5.8 / 11.9 (from 1024 sites per CTA on a thread owns 4 sites; from 2048 the 64-register instance spills).
bool heun_persist_preferred(const Ctx& c) {
  PersistShape sh;
  if (!heun_persist_supported(c) || !persist_shape(c, sh)) return false;
  const int64_t per_cta = (int64_t)sh.ppc * c.d.nz * c.d.ny;
  const bool film_kernel = heun_fast_supported(c);          // else the replayed kernel is the general one, twice as slow
  const int64_t limit = c.d.lattice == ASD_SC ? (film_kernel ? 2048 : 3072) : (film_kernel ? 1024 : 2048);
  return per_cta <= limit;
}

// n Heun steps in one launch; advances c.step.
asd_status launch_heun_persist(Ctx& c, StageParams& sp, int64_t n) {
  PersistShape sh;
  if (!persist_shape(c, sh)) return ASD_EUNSUPPORTED;
  PersistKernel kern = sh.kern;
  if (cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh.smem) != cudaSuccess) {
    cudaGetLastError();
    return ASD_EUNSUPPORTED;
  }
  PersistParams p;
  p.arrays = c.arrays; p.as = (uint32_t)c.as;
  p.oS = (uint32_t)c.aS * p.as; p.oSigma = AR_SIGMA * p.as; p.oB = AR_B * p.as;
  p.col = sp.col; p.grain = sp.grain;
  p.nx = c.d.nx; p.ny = c.d.ny; p.nz = c.d.nz; p.nyp = c.nyp; p.lead = c.lead; p.ppc = sh.ppc;
  p.pbc_x = c.d.pbc[0]; p.pbc_y = c.d.pbc[1]; p.pbc_z = c.d.pbc[2];
  p.j1 = sp.jx[0]; p.j2 = sp.jx[1]; p.j3 = sp.jx[2];
  p.gdt = sp.gdt; p.lambda = sp.lambda; p.scale = sp.scale;
  p.g0 = sp.g0; p.key = sp.key;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)sh.ncta); cfg.blockDim = dim3((unsigned)sh.threads);
  cfg.dynamicSmemBytes = sh.smem; cfg.stream = c.stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)sh.ncta; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  // one launch carries at most 2^20 steps (the loop counter is 32-bit; a launch of that length runs for seconds)
  while (n > 0) {
    const int64_t k = n < (1ll << 20) ? n : (1ll << 20);
    p.step0 = (uint64_t)c.step; p.nsteps = (int32_t)k;
    cudaLaunchKernelEx(&cfg, kern, p);
    ASD_LAUNCH_CHECK(c, "heun steps (persistent cluster)");
    c.step += k;
    n -= k;
  }
  return ASD_OK;
}

}  // namespace asd
