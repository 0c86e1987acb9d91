// asd_heun_fast.cu -- the hot path, film variant: one fused kernel per stochastic-Heun stage for open-boundary
// films whose grains do not touch (every BASELINE film config: >= 1 nm vacant grain boundaries).
//
// Why it needs no masks and no boundary predicates (asd_internal.cuh):
//   * vacant sites hold S = 0, so their bonds drop out of Eq. (2) by themselves; two different grains are never
//     neighbours (checked at create time), so "same grain" never has to be tested;
//   * rows are stored padded with zeros, so y-1 of j = 0 and y+1 of j = ny-1 read zeros with the same unconditional
//     loads as interior sites;
//   * a missing x+-1 or z+-1 row (open window edge) is redirected to the all-zero row by one select per row.
// Each thread owns 4 consecutive sites of one y-row: every neighbour row is one aligned 128-bit load per component,
// the two y-edge sites are scalar loads at immediate offsets from the same address.  All arrays share one base and
// one 32-bit element offset (13 arrays at a common stride).  Noise is generated in registers (asd_rng.cuh).
//
// Bytes per site per stage that must come from / go to HBM: 52; neighbour re-reads are served
// by L1/L2.
#include "asd_internal.cuh"
#include "asd_site.cuh"

namespace asd {

namespace {

constexpr int LAT_SC = 0, LAT_L10 = 1;

struct FastParams {
  const float* arrays;
  float* arrays_w;
  uint32_t as;                     // array stride (elements)
  uint32_t oX, oA, oOut, oOutA;    // element offsets of component 0 of X, A, out, outA (array index * as)
  uint32_t oSigma, oB;
  const uint32_t* col;             // column table at the window origin: grain id + 1 in the low 16 bits (0 = vacant)
  const float4* grain;             // (e_x, e_y, e_z, 2 k_u/mu_s) per grain id + 1; entry 0 = zeros
  uint32_t nthreads, ngrp, nz, nx, ny, nyp, planep, lead;
  uint32_t pf_elems;               // elements of one array spanned by the sites of one CTA (prefetch size)
  uint32_t m_grp, s_grp, m_nz, s_nz;   // magic numbers: t / ngrp and r / nz
  float j1, j2, j3;
  float gdt, lambda, scale;
  uint32_t n_lo, n_hi;
  const DynState* dyn;
  DemagGeom dm;                    // demagnetising field per macrocell; used by the DEMAG instances
  uint32_t dm_my;                  // macrocell edge in y (sites)
  const float* edgeB;              // multiscale window: mesh exchange field on planes 0 / nx-1 (MM instances)
  uint64_t g0;
  PhiloxKey key;
};

// n / d for n < 2^31 (m == 0 means d == 1): q = umulhi(n, m) >> s, m = floor(2^(31+L)/d) + 1, s = L - 1,
// L = ceil(log2 d)  (Granlund-Montgomery round-up method with 31-bit dividends: exact).
__device__ __forceinline__ uint32_t fastdiv(uint32_t n, uint32_t m, uint32_t s) {
  return m ? (__umulhi(n, m) >> s) : n;
}

__device__ __forceinline__ float4 ld4(const float* base, uint32_t e) {
  return __ldg(reinterpret_cast<const float4*>(base + e));
}
__device__ __forceinline__ void st4(float* base, uint32_t e, const float v[4]) {
  *reinterpret_cast<float4*>(base + e) = make_float4(v[0], v[1], v[2], v[3]);
}

// Distance, in units of 256 threads, of the L2 prefetch (see the kernel): a third of a wave of 148 SMs x 768 threads.  Measured on cfg4:
// 64 .. 222 are equivalent (-6 % per stage), 444 gains nothing, 888 and more evict the lines before they are used.
constexpr uint32_t kPrefetchAhead = 148;

// CTA shape: 128 threads x 5 CTAs per SM (96 registers per thread).  Measured on cfg4: 57.9 us per stage, against
// 59.9 (256 x 3, 80 registers), 58.3 (128 x 4), 58.8 (128 x 6), 60.8 (256 x 2), 69.5 (512 x 1).
template <int LAT, int STAGE, int NT = 128, int MINB = 5, bool DEMAG = false, bool MM = false>
__global__ void __launch_bounds__(NT, MINB) heun_stage_fast(const FastParams p) {
  // ---- L2 prefetch: one bulk-prefetch instruction per streamed array brings the sites of the CTA that will run
  // kPrefetchAhead blocks later from HBM into L2.  It holds no registers and nobody waits for it; when that CTA's
  // loads are issued they find their lines in L2 instead of paying the DRAM latency.
  {
    constexpr uint32_t kArr = (STAGE == 0) ? 7u : 10u;           // X(3), sigma, B(3) [, A(3)]
    const uint32_t tb = (blockIdx.x + kPrefetchAhead * 256u / NT) * NT;
    if (threadIdx.x < kArr && tb < p.nthreads) {
      const uint32_t rb = fastdiv(tb, p.m_grp, p.s_grp);
      const uint32_t eb = p.lead + rb * p.nyp + (tb - rb * p.ngrp) * 4u;     // multiple of 4 elements: 16-byte aligned
      const uint32_t a = threadIdx.x;
      const uint32_t off = a < 3u ? p.oX + a * p.as : (a == 3u ? p.oSigma : (a < 7u ? p.oB + (a - 4u) * p.as
                                                                                     : p.oA + (a - 7u) * p.as));
      const uint32_t room = p.as - eb;                           // never past the end of the array
      const uint32_t bytes = ((p.pf_elems < room ? p.pf_elems : room) * 4u) & ~15u;
      if (bytes)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p.arrays + (off + eb)), "r"(bytes) : "memory");
    }
  }
  // Programmatic dependent launch: this grid may be scheduled while the previous kernel of the stream drains; nothing
  // above or below this line up to the wait touches memory that kernel writes (the prefetch only moves lines into L2).
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const uint32_t t = blockIdx.x * NT + threadIdx.x;
  if (t >= p.nthreads) return;
  const uint32_t r = fastdiv(t, p.m_grp, p.s_grp);
  const uint32_t j0 = (t - r * p.ngrp) * 4u;
  const uint32_t i = fastdiv(r, p.m_nz, p.s_nz);
  const uint32_t k = r - i * p.nz;
  const uint32_t e = p.lead + r * p.nyp + j0;                    // own sites
  // neighbour rows; a row outside the window is read from the zero lead (elements [j0+3, j0+8] < lead)
  const uint32_t ez = j0 + 4u;
  const uint32_t e_zp = (k + 1u < p.nz) ? e + p.nyp : ez;
  const uint32_t e_zm = (k > 0u) ? e - p.nyp : ez;
  const uint32_t e_xp = (i + 1u < p.nx) ? e + p.planep : ez;
  const uint32_t e_xm = (i > 0u) ? e - p.planep : ez;

  // every address below is arrays + (one 32-bit element index): a single widening multiply-add per access
  const float* __restrict__ base = p.arrays;
  asm volatile("griddepcontrol.wait;" ::: "memory");           // the previous kernel's stores are complete and visible

  // ---- exchange field, Eq. (2): shell sums first, one multiply per shell ----
  float own[3][6];                // own row with its y-1 and y+1 edge sites
  float Bex[3][4];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const uint32_t oc = p.oX + (uint32_t)c * p.as;
    const float* q_own = base + (oc + e);
    const float* q_xp = base + (oc + e_xp);
    const float* q_xm = base + (oc + e_xm);
    const float4 o = __ldg(reinterpret_cast<const float4*>(q_own));
    own[c][0] = __ldg(q_own - 1); own[c][1] = o.x; own[c][2] = o.y; own[c][3] = o.z; own[c][4] = o.w;
    own[c][5] = __ldg(q_own + 4);
    const float4 zp = ld4(base, oc + e_zp), zm = ld4(base, oc + e_zm);
    const float4 xp = __ldg(reinterpret_cast<const float4*>(q_xp)), xm = __ldg(reinterpret_cast<const float4*>(q_xm));
    const float zs[4] = {zp.x + zm.x, zp.y + zm.y, zp.z + zm.z, zp.w + zm.w};
    if (LAT == LAT_SC) {
      // 6 nearest neighbours, one J
      const float xs[4] = {xp.x + xm.x, xp.y + xm.y, xp.z + xm.z, xp.w + xm.w};
#pragma unroll
      for (int v = 0; v < 4; ++v) Bex[c][v] = p.j1 * ((xs[v] + zs[v]) + (own[c][v] + own[c][v + 2]));
    } else {
      // 4 in-plane nn (J1), 2 out-of-plane (J2), 4 in-plane nnn (J3): "4 nearest + 6 next nearest"
      float xs[6];
      xs[0] = __ldg(q_xp - 1) + __ldg(q_xm - 1);
      xs[1] = xp.x + xm.x; xs[2] = xp.y + xm.y; xs[3] = xp.z + xm.z; xs[4] = xp.w + xm.w;
      xs[5] = __ldg(q_xp + 4) + __ldg(q_xm + 4);
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float s1 = xs[v + 1] + (own[c][v] + own[c][v + 2]);
        const float s3 = xs[v] + xs[v + 2];
        Bex[c][v] = fmaf(p.j3, s3, fmaf(p.j2, zs[v], p.j1 * s1));
      }
    }
  }

  if (MM) {
    // multiscale window: the x neighbours beyond the first / last plane are held mesh directions; their share of
    // Eq. (2) was summed per site at the last exchange (asd_mm.cu) and is added here
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      if (i != (side == 0 ? 0u : p.nx - 1u)) continue;
      const float* eb = p.edgeB + ((uint32_t)side * 3u * p.planep + k * p.nyp + j0);
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float4 ev = __ldg(reinterpret_cast<const float4*>(eb + (uint32_t)c * p.planep));
        Bex[c][0] += ev.x; Bex[c][1] += ev.y; Bex[c][2] += ev.z; Bex[c][3] += ev.w;
      }
    }
  }

  // ---- per-site inputs ----
  const float4 sg4 = ld4(base, p.oSigma + e);
  const float4 bx4 = ld4(base, p.oB + e), by4 = ld4(base, p.oB + p.as + e), bz4 = ld4(base, p.oB + 2u * p.as + e);
  const uint32_t ec = i * p.ny + j0;                             // column (i, j0) of the window
  // Anisotropy parameters (e_x, e_y, e_z, 2 k_u/mu_s): the 4 columns' grain ids (one 128-bit load of the column table)
  // and ONE gather from the per-grain table.  A vacant column (id 0) may borrow its neighbour's parameters: its spins are
  // 0, so its field does nothing.  Two different grains inside one group of 4 sites (grain boundaries of < 3 sites)
  // are flagged in the column table at set-up time and take a per-site gather.
  const uint4 cid4 = __ldg(reinterpret_cast<const uint4*>(p.col + ec));
  const uint32_t gid = max(max(cid4.x & 0xFFFFu, cid4.y & 0xFFFFu), max(cid4.z & 0xFFFFu, cid4.w & 0xFFFFu));
  const bool mixed = (cid4.x & COL_GROUP_MIXED) != 0u;           // set-up flagged this group: rare, divergent path
  // the rare gather sits HERE, before the unrolled site loop: a branch inside that loop would split it into basic blocks
  // and cost the interleaving of the four sites' Philox chains (measured: 57.1 -> 61.4 us per stage)
  float4 gp4[4];
  gp4[0] = gp4[1] = gp4[2] = gp4[3] = __ldg(p.grain + gid);
  if (mixed) {
    gp4[0] = __ldg(p.grain + (cid4.x & 0xFFFFu)); gp4[1] = __ldg(p.grain + (cid4.y & 0xFFFFu));
    gp4[2] = __ldg(p.grain + (cid4.z & 0xFFFFu)); gp4[3] = __ldg(p.grain + (cid4.w & 0xFFFFu));
  }
  const float sg[4] = {sg4.x, sg4.y, sg4.z, sg4.w};
  const float bx[4] = {bx4.x, bx4.y, bx4.z, bx4.w}, by[4] = {by4.x, by4.y, by4.z, by4.w},
              bz[4] = {bz4.x, bz4.y, bz4.z, bz4.w};
  float Ain[3][4];
  if (STAGE == 1) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float4 a = ld4(base, p.oA + (uint32_t)c * p.as + e);
      Ain[c][0] = a.x; Ain[c][1] = a.y; Ain[c][2] = a.z; Ain[c][3] = a.w;
    }
  }

  // ---- noise, torque, update, renormalise ----
  const uint64_t g = p.g0 + (uint64_t)(r * p.ny + j0);           // global site id of the first own site
  uint32_t n_lo = p.n_lo, n_hi = p.n_hi; float scale = p.scale;
  resolve_dyn(p.dyn, n_lo, n_hi, scale);
  const SiteConst sc{p.gdt, p.lambda, scale};
  // the 4 sites lie in at most two macrocells (any my >= 3; for my < 3 the kernel is not used with demag)
  float Bd_lo[3] = {0.0f, 0.0f, 0.0f}, Bd_hi[3] = {0.0f, 0.0f, 0.0f};
  uint32_t dm_split = 0u;                          // sites j < dm_split take Bd_lo
  if (DEMAG) {
    const uint32_t q_lo = demag_cell(p.dm, i, j0, k), q_hi = demag_cell(p.dm, i, j0 + 3u, k);
    dm_split = (q_lo == q_hi) ? 0xFFFFFFFFu : (div_u31(j0 + 3u, p.dm.my_m, p.dm.my_s) * p.dm_my);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      Bd_lo[c] = __ldg(p.dm.B + ((uint32_t)c * p.dm.comp_stride + q_lo));
      Bd_hi[c] = __ldg(p.dm.B + ((uint32_t)c * p.dm.comp_stride + q_hi));
    }
  }
  float o[3][4], oA[3][4];
#pragma unroll
  for (int v = 0; v < 4; ++v) {
    uint32_t rnd[4];
    philox_site(p.key, n_lo, n_hi, g + (uint64_t)v, 0u, rnd);
    float xi[3];
    normals3(rnd, xi);
    const float Xs[3] = {own[0][v + 1], own[1][v + 1], own[2][v + 1]};
    float Be[3] = {Bex[0][v], Bex[1][v], Bex[2][v]};
    if (DEMAG) {                                     // Eq. (7): the field of the site's macrocell
      const float* Bd = (j0 + (uint32_t)v < dm_split) ? Bd_lo : Bd_hi;
      Be[0] += Bd[0]; Be[1] += Bd[1]; Be[2] += Bd[2];
    }
    const float Bap[3] = {bx[v], by[v], bz[v]};
    const float Ai[3] = {Ain[0][v], Ain[1][v], Ain[2][v]};
    float ov[3], oAv[3];
    site_update<STAGE>(sc, Xs, Be, gp4[v], Bap, sg[v], xi, Ai, ov, oAv);
    o[0][v] = ov[0]; o[1][v] = ov[1]; o[2][v] = ov[2];
    if (STAGE == 0) { oA[0][v] = oAv[0]; oA[1][v] = oAv[1]; oA[2][v] = oAv[2]; }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) st4(p.arrays_w, p.oOut + (uint32_t)c * p.as + e, o[c]);
  if (STAGE == 0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) st4(p.arrays_w, p.oOutA + (uint32_t)c * p.as + e, oA[c]);
  }
}


template <int LAT, bool DEMAG, bool MM = false, int NT = 128, int MINB = 5>
asd_status launch_pair_fast(Ctx& c, FastParams& f) {
  const unsigned blocks = (f.nthreads + NT - 1u) / NT;
  f.pf_elems = ((uint32_t)NT * 4u / f.ny + 2u) * f.nyp;
  const uint32_t as = f.as;
  f.oX = (uint32_t)c.aS * as; f.oOut = (uint32_t)c.aSt * as; f.oOutA = AR_A * as; f.oA = AR_A * as;
  if (DEMAG && (c.demag_refresh & 1)) { const asd_status st = launch_demag(c, c.aS); if (st != ASD_OK) return st; }
  launch_pdl(heun_stage_fast<LAT, 0, NT, MINB, DEMAG, MM>, blocks, NT, c.launch_stream, f, c.launch_stream == c.stream);
  ASD_LAUNCH_CHECK(c, "heun predictor (fast)");
  f.oX = (uint32_t)c.aSt * as; f.oOut = (uint32_t)c.aS * as;
  if (DEMAG && (c.demag_refresh & 2)) { const asd_status st = launch_demag(c, c.aSt); if (st != ASD_OK) return st; }
  launch_pdl(heun_stage_fast<LAT, 1, NT, MINB, DEMAG, MM>, blocks, NT, c.launch_stream, f, c.launch_stream == c.stream);
  ASD_LAUNCH_CHECK(c, "heun corrector (fast)");
  return ASD_OK;
}

}  // namespace

// Open boundaries, built-in shells, ny a multiple of 4, grains that do not touch, and 32-bit element offsets.
bool heun_fast_supported(const Ctx& c) {
  return c.d.ell_width == 0 && !c.d.pbc[0] && !c.d.pbc[1] && !c.d.pbc[2] && (c.d.ny % 4 == 0) && !c.grains_touch &&
         (int64_t)AR_COUNT * c.as < (1ll << 31) && c.d.track_nx * (int64_t)c.d.ny < (1ll << 30);
}

asd_status launch_heun_fast(Ctx& c, StageParams& p) {
  FastParams f;
  f.arrays = c.arrays; f.arrays_w = c.arrays; f.as = (uint32_t)c.as;
  f.oSigma = AR_SIGMA * f.as; f.oB = AR_B * f.as;
  f.col = p.col; f.grain = p.grain;
  f.ngrp = (uint32_t)(c.d.ny / 4); f.nthreads = (uint32_t)c.nrows * f.ngrp;
  f.nz = (uint32_t)c.d.nz; f.nx = (uint32_t)c.d.nx; f.ny = (uint32_t)c.d.ny; f.nyp = (uint32_t)c.nyp; f.lead = (uint32_t)c.lead;
  f.planep = (uint32_t)c.d.nz * (uint32_t)c.nyp;
  magic_u31(f.ngrp, f.m_grp, f.s_grp);
  magic_u31(f.nz, f.m_nz, f.s_nz);
  f.j1 = p.jx[0]; f.j2 = p.jx[1]; f.j3 = p.jx[2];
  f.gdt = p.gdt; f.lambda = p.lambda; f.scale = p.scale;
  f.n_lo = p.n_lo; f.n_hi = p.n_hi; f.dyn = p.dyn; f.g0 = p.g0; f.key = p.key;
  f.dm = p.dm; f.dm_my = (uint32_t)c.d.macro[1];
  f.edgeB = p.edgeB;
  if (p.edgeB) {
    if (p.dm.B) return c.d.lattice == ASD_SC ? launch_pair_fast<LAT_SC, true, true>(c, f) : launch_pair_fast<LAT_L10, true, true>(c, f);
    return c.d.lattice == ASD_SC ? launch_pair_fast<LAT_SC, false, true>(c, f) : launch_pair_fast<LAT_L10, false, true>(c, f);
  }
  if (p.dm.B) return c.d.lattice == ASD_SC ? launch_pair_fast<LAT_SC, true>(c, f) : launch_pair_fast<LAT_L10, true>(c, f);
  return c.d.lattice == ASD_SC ? launch_pair_fast<LAT_SC, false>(c, f) : launch_pair_fast<LAT_L10, false>(c, f);
}

}  // namespace asd
