// asd_heun_fused.cu -- the hot path, fused variant: ONE kernel per stochastic-Heun step.
//
// The two-kernel step writes the predictor's S~ and A = S + dt/2 k1 to HBM and reads them back (104 B per site per
// step).  Here the predictor's results never leave the SM: 40 B per site per step -- S in (12),
// sigma and B in (16), S out (12) -- and the noise of a site (Philox4x32-10 + Box-Muller) is generated once per step
// instead of once per stage.
//
// How.  Same lattices as the film kernel (open boundaries, built-in shells, ny % 4 == 0, grains that do not touch; a
// missing or vacant neighbour is a stored or TMA-filled zero, so Eq. (2) needs no mask).  The window is cut into
// y-strips of BY sites and x-chunks of CX planes; one CTA owns one (strip, chunk), holds the whole film thickness and
// MARCHES along x.  Per march step m (predictor plane q, corrector plane q - 1):
//   * S planes q-1, q, q+1 sit in a 4-slot shared-memory ring; plane q+2 is in flight.  One TMA box
//     [3 components][nz + 2 rows][BY + 8 sites] per plane (cp.async.bulk.tensor.4d completing on an mbarrier); rows
//     z = -1, nz, columns y < 0, >= ny and planes x < 0, >= nx are zero-filled by the TMA: the open boundary.
//   * predictor of plane q from the S ring: the "main" threads own 4 consecutive y-sites of one z-row of the strip
//     (same (row, group) for the whole march); the "halo" threads (one warp for nz <= 32) own the two sites of one z-row in the columns next to the
//     strip, whose S~ the strip's corrector needs and which are RECOMPUTED here (the noise is a pure function of
//     (seed, step, global site), so the neighbouring CTA computes the same values).  S~ goes to a second 4-slot ring
//     in shared memory; A and the stage-independent part of the field, sigma xi + s B_app, stay in registers.
//   * one CTA barrier; thread 0 then refills the S slot that has just been read for the last time.
//   * corrector of plane q - 1 from S~ planes q-2, q-1, q; the new S goes to the OTHER spin buffer in HBM (the
//     neighbouring chunk still needs the old values of its halo planes), and the buffers swap roles after the step.
// A chunk recomputes the predictor of one plane before and one after itself (its x halo).
// With four S~ slots one barrier per plane is enough: the predictor of step m+1 writes slot (m+1) % 4, which the
// corrector of step m (slots m-2, m-1, m) does not read, and the predictor of step m+2 is behind the barrier of m+1.
#include <cstdlib>

#include "asd_internal.cuh"
#include "asd_site.cuh"
#include "asd_tma.cuh"

namespace asd {

namespace {

constexpr int LAT_SC = 0, LAT_L10 = 1;
constexpr int kRingS = 4;      // S planes q-1, q, q+1 and the one in flight
constexpr int kRingT = 3;      // S~ planes q-2, q-1, q

struct FusedParams {
  const float* arrays;
  float* arrays_w;
  uint32_t as;                     // array stride (elements)
  int32_t aIn;                     // array index of component 0 of the input spins (TMA coordinate)
  uint32_t oOut, oSigma, oB;       // element offsets (array index * as)
  const uint32_t* col;             // column table at the window origin
  const float4* grain;             // (e_x, e_y, e_z, 2 k_u/mu_s) per grain id + 1
  int32_t nx, ny, nz, nyp, lead;
  int32_t BY, G, nstrips, CX;      // strip width (sites), y-groups per strip row, strips, planes per chunk
  int32_t n_main;                  // threads that own 4-site groups (a multiple of 32); the rest are halo threads
  uint32_t slot_pitch;             // bytes of one ring slot (multiple of 128)
  // Every field term is carried pre-multiplied by -gamma dt / (1 + lambda^2), so that dt f = S x B' + lambda S x (S x B')
  // needs no further scaling: j*s = -gdt J_shell / mu_s, ngdt = -gdt (applied to sigma, B_app and 2 k_u / mu_s on load).
  float j1s, j2s, j3s;
  float ngdt, lambda, scale;
  uint32_t n_lo, n_hi;
  const DynState* dyn;
  uint64_t g0;
  const float* edgeB;              // multiscale window: mesh exchange field on planes 0 / nx-1 ([side][comp][nz*nyp]); nullptr: off
  DemagGeom dm;                    // held demagnetising field per macrocell (DEMAG instances; asd_set_demag_every >= 1)
  uint32_t dm_my;                  // macrocell edge in y (sites)
  // Eq. (6) folded into the corrector (DEMAG instances, dm_acc != nullptr): the new spins' macrocell sums, in units of
  // 1 / dm_fx, are added to dm_acc[comp * comp_stride + cell] -- the layout of dm.B -- for the next refresh of the held field
  long long* dm_acc;
  uint32_t dm_mx, dm_ncyl;         // macrocell edge in x (sites); y-cells a strip can overlap
  float dm_fx;                     // fixed-point scale (a power of two; a whole cell's sum stays below 2^31)
  PhiloxKey key;
};

// dt f(X, B) of Eq. (1) in LL form (asd_site.cuh) from the pre-scaled field B' = -gdt B:  S x B' + lambda S x (S x B')
__device__ __forceinline__ void llg_dt_f(float lambda, const float X[3], float B0, float B1, float B2, float f[3]) {
  const float a0 = X[1] * B2 - X[2] * B1, a1 = X[2] * B0 - X[0] * B2, a2 = X[0] * B1 - X[1] * B0;   // S x B'
  const float b0 = X[1] * a2 - X[2] * a1, b1 = X[2] * a0 - X[0] * a2, b2 = X[0] * a1 - X[1] * a0;   // S x (S x B')
  f[0] = fmaf(lambda, b0, a0);
  f[1] = fmaf(lambda, b1, a1);
  f[2] = fmaf(lambda, b2, a2);
}

// Adds the anisotropy field, Eq. (3), pre-scaled by -gdt, to the exchange field of the 4 sites of a group.  gp = the
// group's (e_x, e_y, e_z, 2 k_u/mu_s), gathered by the caller ahead of time by the group's grain id; a group that holds
// two different grains (rare, flagged at set-up; a branch of its own so that the common path carries no selects)
// gathers per site here.  A vacant site may borrow any parameters: its spin is 0.
__device__ __forceinline__ void add_aniso(const float4* grain, float4 gp, bool mixed, const uint32_t* colp, float ngdt,
                                          const float X[3][4], float Bex[3][4]) {
  if (!mixed) {
    const float kw = gp.w;                             // already pre-scaled by the halo warp
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const float ca = kw * fmaf(X[0][v], gp.x, fmaf(X[1][v], gp.y, X[2][v] * gp.z));
      Bex[0][v] = fmaf(ca, gp.x, Bex[0][v]); Bex[1][v] = fmaf(ca, gp.y, Bex[1][v]); Bex[2][v] = fmaf(ca, gp.z, Bex[2][v]);
    }
  } else {
    const uint4 cc = __ldg(reinterpret_cast<const uint4*>(colp));
    const uint32_t id[4] = {cc.x & 0xFFFFu, cc.y & 0xFFFFu, cc.z & 0xFFFFu, cc.w & 0xFFFFu};
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const float4 gv = __ldg(grain + id[v]);
      const float ca = (ngdt * gv.w) * fmaf(X[0][v], gv.x, fmaf(X[1][v], gv.y, X[2][v] * gv.z));
      Bex[0][v] = fmaf(ca, gv.x, Bex[0][v]); Bex[1][v] = fmaf(ca, gv.y, Bex[1][v]); Bex[2][v] = fmaf(ca, gv.z, Bex[2][v]);
    }
  }
}
// The split barrier of the march: one arrival per warp (release: the warp's shared-memory stores are visible to whoever
// sees the phase complete), waited for later.
__device__ __forceinline__ void warp_arrive(uint32_t bar) {
  __syncwarp();
  if ((threadIdx.x & 31u) == 0u) mbar_arrive(bar);
}
// Counts the warp on a shared-memory counter; true (in lane 0 only) for the warp that comes last, which also resets it.
// Relaxed: used where the warps only have to have CONSUMED something (their loads have returned: the values were used).
__device__ __forceinline__ bool warp_count_last(uint32_t cnt, uint32_t nwarps) {
  __syncwarp();
  bool last = false;
  if ((threadIdx.x & 31u) == 0u) {
    uint32_t old;
    asm volatile("atom.relaxed.cta.shared::cta.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(cnt) : "memory");
    last = (old == nwarps - 1u);
    if (last) asm volatile("st.relaxed.cta.shared::cta.u32 [%0], %1;" ::"r"(cnt), "r"(0u) : "memory");
  }
  return last;
}

__device__ __forceinline__ void red_shared_add(uint32_t a, int v) {
  asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}

constexpr uint32_t kGpRing = 8;   // planes of per-group anisotropy parameters kept in shared memory

// NZ_T / BY_T != 0: film thickness and strip width are compile-time constants (every shared-memory offset becomes an
// immediate of its LDS / STS); 0: taken from the parameter block.
template <int LAT, int NT, int MINB, int NZ_T, int BY_T, bool MM = false, bool DEMAG = false>
__global__ void __launch_bounds__(NT, MINB)
heun_fused(const __grid_constant__ CUtensorMap mapS, const __grid_constant__ CUtensorMap mapF, const FusedParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int NZ = NZ_T ? NZ_T : p.nz, BY = BY_T ? BY_T : p.BY, G = BY / 4;
  const int W = BY + 8, R = NZ + 2;
  const uint32_t rowb = (uint32_t)(W * 4), compb = (uint32_t)(R * W * 4);
  const uint32_t box_bytes = 3u * compb;
  const uint32_t slot_pitch = (NZ_T && BY_T) ? ((box_bytes + 127u) & ~127u) : p.slot_pitch;
  const uint32_t fcomp = (uint32_t)(NZ * BY * 4), fbytes = 4u * fcomp;
  const uint32_t gp_pitch = (uint32_t)((20 * G + 32 + 15) & ~15);   // per plane: float4 per group + 2 halo columns, then one flag word per group
  const uint32_t sm0 = smem_u32(smem_raw);
  const uint32_t bar_full = sm0;                      // S plane landed (TMA transaction count)
  const uint32_t bar_done = sm0 + 32u;                // S~ plane complete
  const uint32_t bar_fld = sm0 + 64u;                 // sigma / B plane landed
  const uint32_t cnt_fld = sm0 + 96u;                 // main warps that have consumed the current sigma / B plane
  const uint32_t gpring = sm0 + 128u;
  const uint32_t sring = gpring + ((kGpRing * gp_pitch + 127u) & ~127u);
  const uint32_t tring = sring + kRingS * slot_pitch;
  const uint32_t fbox = tring + kRingT * slot_pitch;
  // DEMAG with dm_acc: cell sums of the new spins, [2 x-cell parities][3][dm_ncyl][dcz] int32, behind the field box
  const uint32_t sacc = fbox + ((fbytes + 127u) & ~127u);
  const uint32_t acc_comp = DEMAG ? p.dm_ncyl * p.dm.sy * 4u : 0u, acc_buf = 3u * acc_comp;
  const bool acc_on = DEMAG && p.dm_acc != nullptr;

  const int tid = (int)threadIdx.x;
  const int strip = (int)blockIdx.x % p.nstrips, chunk = (int)blockIdx.x / p.nstrips;
  const int j0 = strip * BY;
  const int i0 = chunk * p.CX;
  const int L = min(p.CX, p.nx - i0);                 // planes this CTA updates
  const bool is_main = tid < p.n_main;

  // Anisotropy parameters depend on the column only: for every plane the halo warp looks up, once per 4-site group of the
  // strip, (e_x, e_y, e_z, 2 k_u/mu_s) by the group's grain id (the largest of its 4 columns' ids: vacant columns are 0 and
  // may borrow a neighbour's parameters, their spins are 0) and a flag "this group holds two different grains" (set-up
  // flagged it in the column table; such groups gather per site); lanes G and G + 1 do the same for the two halo columns.
  // Planes i0 - 1 + mm, ring slot mm % 8.  The two dependent table reads of a plane are spread over two march steps
  // (gp_lookup: column entries of plane mm -> packed id; gp_gather: id -> parameters; gp_store: parameters -> ring).
  const int gl = tid - p.n_main;                        // lane of the parameter lookup (halo warp only)
  const int gj = gl < G ? j0 + 4 * gl : (gl == G ? j0 - 1 : j0 + BY);
  auto gp_lookup = [&](int mm) -> uint4 {               // raw column entries (a group's 4, or one halo column's)
    const int plane = i0 - 1 + mm;
    uint4 c4 = make_uint4(0u, 0u, 0u, 0u);
    if (gl < 0 || gl >= G + 2 || plane < 0 || plane >= p.nx || gj < 0 || gj >= p.ny) return c4;
    const uint32_t ci = (uint32_t)plane * (uint32_t)p.ny + (uint32_t)gj;
    if (gl >= G) c4.x = __ldg(p.col + ci) & 0xFFFFu;
    else c4 = __ldg(reinterpret_cast<const uint4*>(p.col + ci));
    return c4;
  };
  auto gp_pack = [&](uint4 cid4) -> uint32_t {          // grain id | bit 31: two grains in the group
    const uint32_t gid = max(max(cid4.x & 0xFFFFu, cid4.y & 0xFFFFu), max(cid4.z & 0xFFFFu, cid4.w & 0xFFFFu));
    return gid | ((cid4.x & COL_GROUP_MIXED) ? 0x80000000u : 0u);
  };
  auto gp_gather = [&](uint32_t cg) -> float4 { return __ldg(p.grain + (cg & 0xFFFFu)); };
  auto gp_store = [&](int mm, uint32_t cg, float4 gp) {
    if (gl >= 0 && gl < G + 2) {
      const uint32_t slot = gpring + ((uint32_t)mm & (kGpRing - 1u)) * gp_pitch;
      sts4(slot + 16u * (uint32_t)gl, gp.x, gp.y, gp.z, gp.w * p.ngdt);      // pre-scaled like every field term
      if (gl < G) sts1(slot + 16u * (uint32_t)(G + 2) + 4u * (uint32_t)gl, __uint_as_float(cg >> 31));
    }
  };

  // S~ ring starts as zeros: the rows z = -1 and z = nz, and the columns of a ragged last strip, are never written.
  for (uint32_t o = (uint32_t)tid * 16u; o < kRingT * slot_pitch; o += (uint32_t)blockDim.x * 16u)
    sts4(tring + o, 0.0f, 0.0f, 0.0f, 0.0f);
  // ... and so does the parameter ring (the corrector of march step 0 reads the slot of a plane nobody fills; its result
  // is discarded, but a stray "two grains" flag would send it to the column table)
  for (uint32_t o = (uint32_t)tid * 16u; o < kGpRing * gp_pitch; o += (uint32_t)blockDim.x * 16u)
    sts4(gpring + o, 0.0f, 0.0f, 0.0f, 0.0f);
  if (acc_on)
    for (uint32_t o = (uint32_t)tid * 4u; o < 2u * acc_buf; o += (uint32_t)blockDim.x * 4u) sts1(sacc + o, 0.0f);
  asm volatile("bar.sync 0;" ::: "memory");
  if (tid == 0) {
    for (int s = 0; s < 4; ++s) {
      mbar_init(bar_full + 8u * s, 1u); mbar_init(bar_done + 8u * s, blockDim.x / 32u);
    }
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(cnt_fld), "r"(0u) : "memory");
    mbar_init(bar_fld, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  // Programmatic dependent launch: everything above overlaps the tail of the previous step's grid; nothing below the
  // wait runs before that grid has completed (it wrote the spins this one reads and read the buffer this one writes).
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("bar.sync 0;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");

  // S ring plane u (u = 0 is window plane i0 - 2) -> slot u % 4;  field plane of march step m = window plane i0 - 1 + m
  auto issue_S = [&](int u) {
    const uint32_t s = (uint32_t)(u & (kRingS - 1));
    mbar_expect_tx(bar_full + 8u * s, box_bytes);
    tma_load_4d(sring + s * slot_pitch, &mapS, bar_full + 8u * s, j0 - 4, -1, i0 - 2 + u, p.aIn);
  };
  auto issue_F = [&](int m) {
    mbar_expect_tx(bar_fld, fbytes);
    tma_load_4d(fbox, &mapF, bar_fld, j0, 0, i0 - 1 + m, AR_SIGMA);
  };
  if (tid == 0) {
    for (int u = 0; u < kRingS; ++u) issue_S(u);       // L >= 1: planes u = 0 .. L+3 are all needed
    issue_F(0);
    for (int m = 1; m <= 3 && m <= L + 1; ++m) tma_prefetch_4d(&mapF, j0, 0, i0 - 1 + m, AR_SIGMA);
  }

  // Parameter ring: planes 0 and 1 of the march directly, plane 2 gathered, plane 3 looked up.  Done after the first
  // TMA loads have been issued, so that these two dependent table reads overlap the flight of the first S planes; the
  // main threads meet the halo warp at named barrier 1 before their first use.
  uint4 cid_next = make_uint4(0u, 0u, 0u, 0u);
  float4 gp_next = make_float4(0.f, 0.f, 1.f, 0.f);
  uint32_t cg_gath = 0u;
  if (!is_main) {
    const uint32_t c0 = gp_pack(gp_lookup(0)), c1 = gp_pack(gp_lookup(1));
    cg_gath = gp_pack(gp_lookup(2)); cid_next = gp_lookup(3);
    const float4 g0 = gp_gather(c0), g1 = gp_gather(c1);
    gp_next = gp_gather(cg_gath);
    gp_store(0, c0, g0); gp_store(1, c1, g1);
  }
  uint32_t n_lo = p.n_lo, n_hi = p.n_hi; float scale = p.scale;
  resolve_dyn(p.dyn, n_lo, n_hi, scale);
  const float sscale = p.ngdt * scale;                // B'_app = sscale * B
  const float lambda = p.lambda;
  const uint32_t planep = (uint32_t)(NZ * p.nyp);
  auto done_bar = [&](int m) { return bar_done + 8u * (uint32_t)(m & 3); };
  auto arrive_done = [&](int m) { warp_arrive(done_bar(m)); };
  auto phase = [](int m) { return (uint32_t)(m >> 2) & 1u; };

  // DEMAG with dm_acc, halo warp(s): the shared sums of the cells with x index ca (absolute) -> global, slots cleared
  auto acc_flush = [&](uint32_t ca) {
    const uint32_t nent = p.dm_ncyl * p.dm.sy, cy0 = div_u31((uint32_t)j0, p.dm.my_m, p.dm.my_s), dcy = p.dm.sx / p.dm.sy;
    const uint32_t sb = sacc + (ca & 1u) * acc_buf;
    for (uint32_t t = (uint32_t)(tid - p.n_main); t < 3u * nent; t += blockDim.x - (uint32_t)p.n_main) {
      const uint32_t comp = t / nent, r = t - comp * nent, cyl = r / p.dm.sy, ck = r - cyl * p.dm.sy;
      const int v = __float_as_int(lds1(sb + t * 4u));
      if (v != 0 && cy0 + cyl < dcy) {
        atomicAdd(reinterpret_cast<unsigned long long*>(p.dm_acc) +
                      (comp * p.dm.comp_stride + (ca - p.dm.c0) * p.dm.sx + (cy0 + cyl) * p.dm.sy + ck),
                  (unsigned long long)(long long)v);
        sts1(sb + t * 4u, 0.0f);
      }
    }
  };

  if (is_main) {
    // ================= main threads: 4 consecutive y-sites of one z-row, predictor and corrector =================
    const int k = tid / G, g = tid - k * G;
    const int j = j0 + 4 * g;
    const bool active = (k < NZ) && (j < p.ny);
    // own float4 inside component 0 of a slot (inactive threads read a valid dummy position and write nothing)
    const uint32_t own_b = active ? (uint32_t)(((k + 1) * W + 4 + 4 * g) * 4) : (uint32_t)((W + 4) * 4);
    const uint32_t fown = fbox + (active ? (uint32_t)((k * BY + 4 * g) * 4) : 0u);
    const uint32_t gown = gpring + 16u * (uint32_t)g, gflag = gpring + 16u * (uint32_t)(G + 2) + 4u * (uint32_t)g;
    // element of the group in predictor plane q = i0 - 1 (wraps below zero for q = -1; not dereferenced then)
    uint32_t e = (uint32_t)(p.lead + ((i0 - 1) * NZ + k) * p.nyp + j);
    uint32_t ec = (uint32_t)((i0 - 1) * p.ny + j);                      // column (q, j) of the window
    uint64_t gsite = p.g0 + (uint64_t)(int64_t)(((int64_t)(i0 - 1) * NZ + k) * p.ny + j);
    const uint32_t gplane = (uint32_t)(NZ * p.ny);

    // carried from the predictor of plane q to its corrector one march step later
    float A[3][4], Bs[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int v = 0; v < 4; ++v) { A[c][v] = 0.0f; Bs[c][v] = 0.0f; }
    // L1_0 only: the y-1 / y+4 edge columns of the group's row are 16-byte-strided scalar reads (4 shared-memory
    // wavefronts each); every plane's pair is read once and kept while the plane is the x+1, own and x-1 plane.
    float sP[3][2], sC[3][2];      // S edges of planes q-1, q
    float tP[3][2], tC[3][2];      // S~ edges of planes q-2, q-1
#pragma unroll
    for (int c = 0; c < 3; ++c) { sP[c][0] = sP[c][1] = sC[c][0] = sC[c][1] = tP[c][0] = tP[c][1] = tC[c][0] = tC[c][1] = 0.0f; }

    // held demagnetising field (DEMAG): the thread's two macrocells across the film and through its thickness are fixed
    uint32_t dm_yz_lo = 0u, dm_yz_hi = 0u;
    int dm_nlo = 4;                                    // own sites v < dm_nlo lie in the lower-y cell
    uint32_t sacc_own = sacc;                          // the lower-y cell's slot in the shared cell sums (parity 0, component 0)
    if (DEMAG && active) {
      const uint32_t cj_lo = div_u31((uint32_t)j, p.dm.my_m, p.dm.my_s), cj_hi = div_u31((uint32_t)j + 3u, p.dm.my_m, p.dm.my_s);
      const uint32_t ck = div_u31((uint32_t)k, p.dm.mz_m, p.dm.mz_s);
      dm_yz_lo = cj_lo * p.dm.sy + ck; dm_yz_hi = cj_hi * p.dm.sy + ck;
      dm_nlo = (cj_lo == cj_hi) ? 4 : (int)(cj_hi * p.dm_my) - j;
      sacc_own = sacc + ((cj_lo - div_u31((uint32_t)j0, p.dm.my_m, p.dm.my_s)) * p.dm.sy + ck) * 4u;
    }
    mbar_wait_long(bar_full + 0u, 0u);
    mbar_wait_long(bar_full + 8u, 0u);
    asm volatile("bar.sync 1;" ::: "memory");          // the parameter ring's first planes are in place
    if (LAT == LAT_L10) {
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const uint32_t a0 = sring + own_b + (uint32_t)c * compb, a1 = a0 + slot_pitch;
        sP[c][0] = lds1(a0 - 4u); sP[c][1] = lds1(a0 + 16u);
        sC[c][0] = lds1(a1 - 4u); sC[c][1] = lds1(a1 + 16u);
      }
    }
    uint32_t t3 = 0u;                                  // m % 3: S~ slot of plane q

    for (int m = 0; m <= L + 1; ++m) {
      const uint32_t tN = tring + t3 * slot_pitch + own_b;                                   // S~ plane q
      const uint32_t tCs = tring + (t3 == 0u ? 2u : t3 - 1u) * slot_pitch + own_b;           // q - 1
      const uint32_t tPs = tring + (t3 == 2u ? 0u : t3 + 1u) * slot_pitch + own_b;           // q - 2
      mbar_wait_long(bar_full + 8u * (uint32_t)((m + 2) & (kRingS - 1)), phase(m + 2));      // S plane q + 1

      // ---- predictor of plane q: S~ = normalise(S + dt k1), A = S + dt/2 k1 ----
      float An[3][4], Bn[3][4];                        // this plane's A and -gdt (sigma xi + s B_app)
      {
        const uint32_t prev = sring + (uint32_t)(m & 3) * slot_pitch + own_b;
        const uint32_t cur = sring + (uint32_t)((m + 1) & 3) * slot_pitch + own_b;
        const uint32_t next = sring + (uint32_t)((m + 2) & 3) * slot_pitch + own_b;
        float X[3][4], Bex[3][4];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const uint32_t cb = (uint32_t)c * compb;
          const float4 o = lds4(cur + cb);
          const float4 zp = lds4(cur + cb + rowb), zm = lds4(cur + cb - rowb);
          const float4 xp = lds4(next + cb), xm = lds4(prev + cb);
          X[c][0] = o.x; X[c][1] = o.y; X[c][2] = o.z; X[c][3] = o.w;
          const float zs[4] = {zp.x + zm.x, zp.y + zm.y, zp.z + zm.z, zp.w + zm.w};
          if (LAT == LAT_SC) {
            // 6 nearest neighbours, one J
            const float own[6] = {lds1(cur + cb - 4u), o.x, o.y, o.z, o.w, lds1(cur + cb + 16u)};
            const float xs[4] = {xp.x + xm.x, xp.y + xm.y, xp.z + xm.z, xp.w + xm.w};
#pragma unroll
            for (int v = 0; v < 4; ++v) Bex[c][v] = p.j1s * ((xs[v] + zs[v]) + (own[v] + own[v + 2]));
          } else {
            // 4 in-plane nn (J1), 2 out-of-plane (J2), 4 in-plane nnn (J3): "4 nearest + 6 next nearest"
            const float nL = lds1(next + cb - 4u), nR = lds1(next + cb + 16u);
            const float own[6] = {sC[c][0], o.x, o.y, o.z, o.w, sC[c][1]};
            const float xs[6] = {nL + sP[c][0], xp.x + xm.x, xp.y + xm.y, xp.z + xm.z, xp.w + xm.w, nR + sP[c][1]};
#pragma unroll
            for (int v = 0; v < 4; ++v) {
              const float s1 = xs[v + 1] + (own[v] + own[v + 2]);
              const float s3 = xs[v] + xs[v + 2];
              Bex[c][v] = fmaf(p.j3s, s3, fmaf(p.j2s, zs[v], p.j1s * s1));
            }
            sP[c][0] = sC[c][0]; sP[c][1] = sC[c][1]; sC[c][0] = nL; sC[c][1] = nR;
          }
        }
        {
          const uint32_t gs = ((uint32_t)m & (kGpRing - 1u)) * gp_pitch;
          add_aniso(p.grain, lds4(gown + gs), __float_as_uint(lds1(gflag + gs)) != 0u, p.col + ec, p.ngdt, X, Bex);
        }
        // ---- noise: one Philox block per site per STEP; sigma and B of the plane come from the staged field box ----
        mbar_wait_long(bar_fld, (uint32_t)m & 1u);
        {
          const float4 sg4 = lds4(fown), bx4 = lds4(fown + fcomp), by4 = lds4(fown + 2u * fcomp), bz4 = lds4(fown + 3u * fcomp);
          const float sg[4] = {sg4.x, sg4.y, sg4.z, sg4.w};
          const float bx[4] = {bx4.x, bx4.y, bx4.z, bx4.w}, by[4] = {by4.x, by4.y, by4.z, by4.w},
                      bz[4] = {bz4.x, bz4.y, bz4.z, bz4.w};
          uint32_t rnd[4][4];
          float xi[4][3];
#pragma unroll
          for (int v = 0; v < 4; ++v) philox_site(p.key, n_lo, n_hi, gsite + (uint64_t)v, 0u, rnd[v]);
          normals3_multi<4>(rnd, xi);
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            const float sgs = p.ngdt * sg[v];
            Bn[0][v] = fmaf(sgs, xi[v][0], sscale * bx[v]);
            Bn[1][v] = fmaf(sgs, xi[v][1], sscale * by[v]);
            Bn[2][v] = fmaf(sgs, xi[v][2], sscale * bz[v]);
          }
        }
        if (DEMAG) {
          // Eq. (7), held-field scheme (D3, asd_set_demag_every >= 1): the field of the site's macrocell was
          // computed from S before this step and serves both stages, so it rides with the stage-independent part.  The
          // 4 sites lie in at most two macrocells (my >= 3).
          // Only the x index of the cell changes along the march; the two cells' y-z offsets are per-thread constants.
          // The six values are loaded here, at their point of use (a few-KB table: L1 hits), so that nothing extra is
          // live across the Philox / Box-Muller chains above.
          const int q = i0 - 1 + m;
          if (active && q >= 0 && q < p.nx) {
            const uint32_t cb = (div_u31(p.dm.x0 + (uint32_t)q, p.dm.mx_m, p.dm.mx_s) - p.dm.c0) * p.dm.sx;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              const float lo = p.ngdt * __ldg(p.dm.B + ((uint32_t)c * p.dm.comp_stride + cb + dm_yz_lo));
              const float hi = p.ngdt * __ldg(p.dm.B + ((uint32_t)c * p.dm.comp_stride + cb + dm_yz_hi));
#pragma unroll
              for (int v = 0; v < 4; ++v) Bn[c][v] += (v < dm_nlo) ? lo : hi;
            }
          }
        }
        if (MM) {
          // multiscale window: the held mesh directions beyond the first / last plane enter Eq. (2) of BOTH stages as a
          // constant field, so they ride with the stage-independent part (asd_mm.cu)
          const int q = i0 - 1 + m;
#pragma unroll 1
          for (int side = 0; side < 2; ++side) {
            if (!active || q != (side == 0 ? 0 : p.nx - 1)) continue;
            const float* eb = p.edgeB + ((uint32_t)side * 3u * planep + (uint32_t)(k * p.nyp + j));
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              const float4 ev = __ldg(reinterpret_cast<const float4*>(eb + (uint32_t)c * planep));
              Bn[c][0] = fmaf(p.ngdt, ev.x, Bn[c][0]); Bn[c][1] = fmaf(p.ngdt, ev.y, Bn[c][1]);
              Bn[c][2] = fmaf(p.ngdt, ev.z, Bn[c][2]); Bn[c][3] = fmaf(p.ngdt, ev.w, Bn[c][3]);
            }
          }
        }
        // the field box is refilled as soon as the last main warp has its values in registers (mid-predictor): the copy
        // has the rest of the march step to land.  That warp issues it.
        if (warp_count_last(cnt_fld, (uint32_t)p.n_main / 32u) && m + 1 <= L + 1) {
          issue_F(m + 1);
          if (m + 4 <= L + 1) tma_prefetch_4d(&mapF, j0, 0, i0 - 1 + m + 4, AR_SIGMA);
        }
        float St[3][4];
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float Xs[3] = {X[0][v], X[1][v], X[2][v]};
          float f[3];
          llg_dt_f(lambda, Xs, Bex[0][v] + Bn[0][v], Bex[1][v] + Bn[1][v], Bex[2][v] + Bn[2][v], f);
          An[0][v] = fmaf(0.5f, f[0], Xs[0]); An[1][v] = fmaf(0.5f, f[1], Xs[1]); An[2][v] = fmaf(0.5f, f[2], Xs[2]);
          float o[3];
          normalise3(Xs[0] + f[0], Xs[1] + f[1], Xs[2] + f[2], o);
          St[0][v] = o[0]; St[1][v] = o[1]; St[2][v] = o[2];
        }
        // a plane outside the window has S = 0 everywhere (TMA fill), hence S~ = 0: the open boundary in x
        if (active) {
#pragma unroll
          for (int c = 0; c < 3; ++c) sts4(tN + (uint32_t)c * compb, St[c][0], St[c][1], St[c][2], St[c][3]);
        }
      }
      arrive_done(m);                                  // this warp's share of S~ plane q is written

      // ---- corrector of plane q - 1, first part: everything that does not need S~ plane q ----
      const bool do_corr = active && (m >= 2);
      float X[3][4], Bp[3][4];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const uint32_t cb = (uint32_t)c * compb;
        const float4 o = lds4(tCs + cb);
        const float4 zp = lds4(tCs + cb + rowb), zm = lds4(tCs + cb - rowb);
        const float4 xm = lds4(tPs + cb);
        X[c][0] = o.x; X[c][1] = o.y; X[c][2] = o.z; X[c][3] = o.w;
        const float zs[4] = {zp.x + zm.x, zp.y + zm.y, zp.z + zm.z, zp.w + zm.w};
        if (LAT == LAT_SC) {
          const float own[6] = {lds1(tCs + cb - 4u), o.x, o.y, o.z, o.w, lds1(tCs + cb + 16u)};
          const float xmv[4] = {xm.x, xm.y, xm.z, xm.w};
#pragma unroll
          for (int v = 0; v < 4; ++v) Bp[c][v] = p.j1s * ((xmv[v] + zs[v]) + (own[v] + own[v + 2]));
        } else {
          const float own[6] = {tC[c][0], o.x, o.y, o.z, o.w, tC[c][1]};
          const float xmv[6] = {tP[c][0], xm.x, xm.y, xm.z, xm.w, tP[c][1]};
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            const float s1 = xmv[v + 1] + (own[v] + own[v + 2]);
            const float s3 = xmv[v] + xmv[v + 2];
            Bp[c][v] = fmaf(p.j3s, s3, fmaf(p.j2s, zs[v], p.j1s * s1));
          }
        }
      }
      {
        const uint32_t gs = ((uint32_t)(m - 1) & (kGpRing - 1u)) * gp_pitch;
        add_aniso(p.grain, lds4(gown + gs), __float_as_uint(lds1(gflag + gs)) != 0u, p.col + (ec - (uint32_t)p.ny), p.ngdt, X, Bp);
      }
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int v = 0; v < 4; ++v) Bp[c][v] += Bs[c][v];

      mbar_wait_long(done_bar(m), phase(m));           // S~ plane q complete; S plane q - 1 is free
      if (tid == 0 && m + kRingS <= L + 3) issue_S(m + kRingS);

      // ---- second part: the x+1 plane, torque, update, store ----
      {
        float So[3][4];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const uint32_t cb = (uint32_t)c * compb;
          const float4 xp = lds4(tN + cb);
          if (LAT == LAT_SC) {
            Bp[c][0] = fmaf(p.j1s, xp.x, Bp[c][0]); Bp[c][1] = fmaf(p.j1s, xp.y, Bp[c][1]);
            Bp[c][2] = fmaf(p.j1s, xp.z, Bp[c][2]); Bp[c][3] = fmaf(p.j1s, xp.w, Bp[c][3]);
          } else {
            const float nL = lds1(tN + cb - 4u), nR = lds1(tN + cb + 16u);
            const float xpv[6] = {nL, xp.x, xp.y, xp.z, xp.w, nR};
#pragma unroll
            for (int v = 0; v < 4; ++v) Bp[c][v] = fmaf(p.j1s, xpv[v + 1], fmaf(p.j3s, xpv[v] + xpv[v + 2], Bp[c][v]));
            tP[c][0] = tC[c][0]; tP[c][1] = tC[c][1]; tC[c][0] = nL; tC[c][1] = nR;
          }
        }
        if (do_corr) {
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            const float Xs[3] = {X[0][v], X[1][v], X[2][v]};
            float f[3];
            llg_dt_f(lambda, Xs, Bp[0][v], Bp[1][v], Bp[2][v], f);
            float o[3];
            normalise3(fmaf(0.5f, f[0], A[0][v]), fmaf(0.5f, f[1], A[1][v]), fmaf(0.5f, f[2], A[2][v]), o);
            So[0][v] = o[0]; So[1][v] = o[1]; So[2][v] = o[2];
          }
          const uint32_t eo = e - planep;              // plane q - 1
#pragma unroll
          for (int c = 0; c < 3; ++c)
            *reinterpret_cast<float4*>(p.arrays_w + (p.oOut + (uint32_t)c * p.as + eo)) =
                make_float4(So[c][0], So[c][1], So[c][2], So[c][3]);
          if (acc_on) {
            // Eq. (6) for the next refresh of the held field: this plane's share of the thread's one or two macrocells,
            // as integers (the sum is then independent of the order in which the threads arrive)
            const uint32_t cpar = div_u31(p.dm.x0 + (uint32_t)(i0 + m - 2), p.dm.mx_m, p.dm.mx_s) & 1u;
            const uint32_t sb = sacc_own + cpar * acc_buf;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              float lo = 0.0f, hi = 0.0f;
#pragma unroll
              for (int v = 0; v < 4; ++v) { if (v < dm_nlo) lo += So[c][v]; else hi += So[c][v]; }
              red_shared_add(sb + (uint32_t)c * acc_comp, __float2int_rn(lo * p.dm_fx));
              if (dm_nlo < 4) red_shared_add(sb + (uint32_t)c * acc_comp + p.dm.sy * 4u, __float2int_rn(hi * p.dm_fx));
            }
          }
        }
      }
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int v = 0; v < 4; ++v) { A[c][v] = An[c][v]; Bs[c][v] = Bn[c][v]; }
      e += planep; ec += (uint32_t)p.ny; gsite += gplane;
      t3 = (t3 == 2u) ? 0u : t3 + 1u;
    }
    if (acc_on) arrive_done(L + 2);                   // the last planes' cell sums are in shared memory
  } else {
    // ================= halo warp(s): the two sites (y = j0 - 1, y = j0 + BY) of one z-row, predictor only; =================
    // ================= and the per-group anisotropy parameters two planes ahead                              =================
    // Lanes of a warp read the same column of different rows (a bank-conflicted pattern), so each halo thread keeps
    // the three columns around its sites for planes q-1, q in registers and loads only plane q+1's and the z
    // neighbours of plane q per march step.
    const float* __restrict__ base = p.arrays;
    const int k = tid - p.n_main;
    const bool row_ok = k < NZ;
    const int jh[2] = {j0 - 1, j0 + BY};
    const bool act[2] = {row_ok && jh[0] >= 0, row_ok && jh[1] < p.ny};
    const int kk = row_ok ? k : 0;
    const uint32_t own_b[2] = {(uint32_t)(((kk + 1) * W + 3) * 4), (uint32_t)(((kk + 1) * W + 4 + BY) * 4)};
    uint32_t e = (uint32_t)(p.lead + ((i0 - 1) * NZ + k) * p.nyp);          // + jh
    uint32_t ec = (uint32_t)((i0 - 1) * p.ny);
    uint64_t gsite = p.g0 + (uint64_t)(int64_t)(((int64_t)(i0 - 1) * NZ + k) * p.ny);
    const uint32_t gplane = (uint32_t)(NZ * p.ny);

    asm volatile("bar.sync 1;" ::: "memory");          // planes 0, 1 of the parameter ring are stored
    mbar_wait_long(bar_full + 0u, 0u);
    mbar_wait_long(bar_full + 8u, 0u);
    // window: rP = plane q-1, rC = plane q; [side][component][column y-1, y, y+1]
    float rP[2][3][3], rC[2][3][3];
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          const uint32_t off = own_b[s] + (uint32_t)c * compb + (uint32_t)(4 * d) - 4u;
          rP[s][c][d] = lds1(sring + off);
          rC[s][c][d] = lds1(sring + slot_pitch + off);
        }
    uint32_t t3 = 0u;
    uint32_t hd_ci[2] = {0xFFFFFFFFu, 0xFFFFFFFFu};     // DEMAG: cell x index whose field hd[] holds, per side
    float hd[2][3] = {{0.0f, 0.0f, 0.0f}, {0.0f, 0.0f, 0.0f}};

    for (int m = 0; m <= L + 1; ++m) {
      const int q = i0 - 1 + m;
      const bool qin = (q >= 0) && (q < p.nx);
      float sg[2] = {0.f, 0.f}, bx[2] = {0.f, 0.f}, by[2] = {0.f, 0.f}, bz[2] = {0.f, 0.f};
#pragma unroll
      for (int s = 0; s < 2; ++s)
        if (act[s] && qin) {
          const uint32_t es = e + (uint32_t)jh[s];
          sg[s] = ldg_stream1(base + (p.oSigma + es));
          bx[s] = ldg_stream1(base + (p.oB + es));
          by[s] = ldg_stream1(base + (p.oB + p.as + es));
          bz[s] = ldg_stream1(base + (p.oB + 2u * p.as + es));
        }
      // parameter ring: plane m + 2 (gathered during the previous march step) goes to slot (m + 2) % 8, last read in
      // march step m - 5; plane m + 3 is gathered, plane m + 4 looked up
      asm volatile("" : "+r"(cid_next.x), "+r"(cid_next.y), "+r"(cid_next.z), "+r"(cid_next.w), "+f"(gp_next.x),
                   "+f"(gp_next.y), "+f"(gp_next.z), "+f"(gp_next.w)::"memory");   // first use of last step's loads: here, not earlier
      gp_store(m + 2, cg_gath, gp_next);
      cg_gath = gp_pack(cid_next);
      gp_next = gp_gather(cg_gath);
      cid_next = gp_lookup(m + 4);
      mbar_wait_long(bar_full + 8u * (uint32_t)((m + 2) & (kRingS - 1)), phase(m + 2));
      const uint32_t cur = sring + (uint32_t)((m + 1) & 3) * slot_pitch, next = sring + (uint32_t)((m + 2) & 3) * slot_pitch;
      const uint32_t tslot = tring + t3 * slot_pitch;
      float rN[2][3][3];
      float o[2][3];
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        float zs[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const uint32_t off = own_b[s] + (uint32_t)c * compb;
#pragma unroll
          for (int d = 0; d < 3; ++d) rN[s][c][d] = lds1(next + off + (uint32_t)(4 * d) - 4u);
          zs[c] = lds1(cur + off + rowb) + lds1(cur + off - rowb);
        }
        o[s][0] = o[s][1] = o[s][2] = 0.0f;
        if (act[s] && qin) {
          uint32_t rnd[4];
          philox_site(p.key, n_lo, n_hi, gsite + (uint64_t)(int64_t)jh[s], 0u, rnd);
          float xi[3];
          normals3(rnd, xi);
          float Xs[3], Bex[3];
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            Xs[c] = rC[s][c][1];
            const float ys = rC[s][c][0] + rC[s][c][2];
            const float xs = rN[s][c][1] + rP[s][c][1];
            if (LAT == LAT_SC) {
              Bex[c] = p.j1s * ((xs + zs[c]) + ys);
            } else {
              const float s3 = (rN[s][c][0] + rP[s][c][0]) + (rN[s][c][2] + rP[s][c][2]);
              Bex[c] = fmaf(p.j3s, s3, fmaf(p.j2s, zs[c], p.j1s * (xs + ys)));
            }
          }
          if (DEMAG) {
            const uint32_t ci = div_u31(p.dm.x0 + (uint32_t)q, p.dm.mx_m, p.dm.mx_s) - p.dm.c0;
            if (ci != hd_ci[s]) {
              hd_ci[s] = ci;
              const uint32_t cq = ci * p.dm.sx + div_u31((uint32_t)jh[s], p.dm.my_m, p.dm.my_s) * p.dm.sy +
                                  div_u31((uint32_t)k, p.dm.mz_m, p.dm.mz_s);
#pragma unroll
              for (int c = 0; c < 3; ++c) hd[s][c] = p.ngdt * __ldg(p.dm.B + ((uint32_t)c * p.dm.comp_stride + cq));
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) Bex[c] += hd[s][c];
          }
          if (MM) {
#pragma unroll 1
            for (int side = 0; side < 2; ++side) {
              if (q != (side == 0 ? 0 : p.nx - 1)) continue;
              const float* eb = p.edgeB + ((uint32_t)side * 3u * planep + (uint32_t)(k * p.nyp + jh[s]));
#pragma unroll
              for (int c = 0; c < 3; ++c) Bex[c] = fmaf(p.ngdt, __ldg(eb + (uint32_t)c * planep), Bex[c]);
            }
          }
          const float4 gp = lds4(gpring + ((uint32_t)m & (kGpRing - 1u)) * gp_pitch + 16u * (uint32_t)(G + s));
          const float ca = gp.w * fmaf(Xs[0], gp.x, fmaf(Xs[1], gp.y, Xs[2] * gp.z));
          const float sgs = p.ngdt * sg[s];
          float f[3];
          llg_dt_f(lambda, Xs, fmaf(ca, gp.x, Bex[0]) + fmaf(sgs, xi[0], sscale * bx[s]),
                   fmaf(ca, gp.y, Bex[1]) + fmaf(sgs, xi[1], sscale * by[s]),
                   fmaf(ca, gp.z, Bex[2]) + fmaf(sgs, xi[2], sscale * bz[s]), f);
          normalise3(Xs[0] + f[0], Xs[1] + f[1], Xs[2] + f[2], o[s]);
        }
      }
      // S~ slot m % 3 held plane q - 3.  Its halo columns were last read by main threads in march step m - 3 (L1_0: as
      // the edges of their x+1 plane) or m - 2 (SC: as the edges of their own plane), i.e. before they arrived for
      // step m - 1.
      if (m >= 1) mbar_wait_long(done_bar(m - 1), phase(m - 1));
      if (acc_on && m >= 4) {
        // every main warp has arrived for step m - 1, i.e. has added plane i0 + m - 4 (corrected in step m - 2) to the cell
        // sums: if that plane closes its macrocell, the cell's sums go to global memory and its slots are cleared (the
        // slots of this parity are next written for the cell after the next, behind this warp's arrival for step m)
        const uint32_t xg = p.dm.x0 + (uint32_t)(i0 + m - 4), ca = div_u31(xg, p.dm.mx_m, p.dm.mx_s);
        if (xg + 1u == (ca + 1u) * p.dm_mx) acc_flush(ca);
      }
#pragma unroll
      for (int s = 0; s < 2; ++s)
        if (act[s]) {
#pragma unroll
          for (int c = 0; c < 3; ++c) sts1(tslot + own_b[s] + (uint32_t)c * compb, o[s][c]);
        }
      arrive_done(m);
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
          for (int d = 0; d < 3; ++d) { rP[s][c][d] = rC[s][c][d]; rC[s][c][d] = rN[s][c][d]; }
      e += planep; ec += (uint32_t)p.ny; gsite += gplane;
      t3 = (t3 == 2u) ? 0u : t3 + 1u;
    }
    if (acc_on) {
      // what is left: the (at most two) cells that the chunk's last two planes belong to
      arrive_done(L + 2);
      mbar_wait_long(done_bar(L + 2), phase(L + 2));
      const uint32_t ca = div_u31(p.dm.x0 + (uint32_t)(i0 + L - 1), p.dm.mx_m, p.dm.mx_s);
      acc_flush(ca);
      if (ca > p.dm.c0) acc_flush(ca - 1u);
    }
  }
}

typedef void (*FusedKernel)(const CUtensorMap, const CUtensorMap, const FusedParams);

// Compiled CTA shapes (threads, CTAs per SM -> register budget): 256 x 2 -> 128 registers (4 warps per scheduler),
// 512 x 1 -> 128.
struct Shape { int nt, minb; };
constexpr Shape kShapes[] = {{256, 2}, {512, 1}};
constexpr int kNumShapes = 2;

// Film thickness 27 planes with 32-site strips (BASELINE configs 1, 3, 4) has its own instance with compile-time shared-
// memory offsets; everything else takes the generic one.
FusedKernel kernel_for(int lattice, int shape, int nz, int by, bool mm = false, bool demag = false) {
  if (demag) {                                          // held demagnetising field: the 256 x 2 shape only
    if (shape != 0) return nullptr;
    if (mm) {                                           // ... with meshes / track-coupled ends as well
      if (nz == 27 && by == 32)
        return lattice == ASD_SC ? heun_fused<LAT_SC, 256, 2, 27, 32, true, true> : heun_fused<LAT_L10, 256, 2, 27, 32, true, true>;
      return lattice == ASD_SC ? heun_fused<LAT_SC, 256, 2, 0, 0, true, true> : heun_fused<LAT_L10, 256, 2, 0, 0, true, true>;
    }
    if (nz == 27 && by == 32)
      return lattice == ASD_SC ? heun_fused<LAT_SC, 256, 2, 27, 32, false, true> : heun_fused<LAT_L10, 256, 2, 27, 32, false, true>;
    return lattice == ASD_SC ? heun_fused<LAT_SC, 256, 2, 0, 0, false, true> : heun_fused<LAT_L10, 256, 2, 0, 0, false, true>;
  }
  if (mm) {                                             // multiscale window: the 256 x 2 shape only
    if (shape != 0) return nullptr;
    if (nz == 27 && by == 32)
      return lattice == ASD_SC ? heun_fused<LAT_SC, 256, 2, 27, 32, true> : heun_fused<LAT_L10, 256, 2, 27, 32, true>;
    return lattice == ASD_SC ? heun_fused<LAT_SC, 256, 2, 0, 0, true> : heun_fused<LAT_L10, 256, 2, 0, 0, true>;
  }
  if (shape == 0 && nz == 27 && by == 32)
    return lattice == ASD_SC ? heun_fused<LAT_SC, 256, 2, 27, 32> : heun_fused<LAT_L10, 256, 2, 27, 32>;
  if (lattice == ASD_SC) return shape == 0 ? heun_fused<LAT_SC, 256, 2, 0, 0> : heun_fused<LAT_SC, 512, 1, 0, 0>;
  return shape == 0 ? heun_fused<LAT_L10, 256, 2, 0, 0> : heun_fused<LAT_L10, 512, 1, 0, 0>;
}

inline int round_up32(int v) { return (v + 31) / 32 * 32; }

uint32_t plan_smem(int nz, int by, uint32_t& slot_pitch) {
  slot_pitch = (uint32_t)align_up((size_t)3 * (nz + 2) * (by + 8) * 4, 128);
  return 128u + (uint32_t)align_up((size_t)kGpRing * (size_t)((20 * (by / 4) + 32 + 15) & ~15), 128) + (kRingS + kRingT) * slot_pitch +
         (uint32_t)align_up((size_t)4 * nz * by * 4, 128);
}

}  // namespace

struct FusedPlan {
  CUtensorMap mapS, mapF;
  FusedKernel kern = nullptr;
  FusedKernel kern_mm = nullptr;   // the instance that adds the mesh exchange field on planes 0 / nx-1 (asd_mm.cu); may be null
  FusedKernel kern_dm = nullptr;   // the instance that adds a held demagnetising field per macrocell; may be null
  FusedKernel kern_dm_mm = nullptr;   // ... and the edge field as well; may be null
  int32_t BY = 0, G = 0, nstrips = 0, CX = 0, nchunks = 0, threads = 0, n_main = 0, ctas_per_sm = 0;
  uint32_t slot_pitch = 0, smem_bytes = 0;
  uint32_t smem_bytes_dm = 0;      // kern_dm: + the shared cell sums of the Eq. (6) epilogue (0: they do not fit; no epilogue)
  uint32_t dm_ncyl = 0;
};

bool heun_fused_supported(const Ctx& c) { return heun_fast_supported(c) && c.d.nz + 2 <= 256; }

// ASD_KERNEL_AUTO takes the fused step for windows of more than 1.5 M sites that give every CTA a march of at least 8
// planes (a chunk recomputes the predictor of 2 extra planes).  Smaller films are L2-resident or launch-bound; there the
// two stage kernels (or their graph replay) stay in charge.  Measured (B200, G updates/s, two-kernel -> fused): cfg4
// 46.0 -> 55.3, cfg3 42.9 -> 46.6, the 336 x 200 x 27 multiscale window (1.81 M sites, 8-plane marches) 39.0 -> 43.8;
// cfg2 46.6 -> 32.3 and cfg1 48.9 -> 41.3 (1 M sites, marches of 5-6 planes).
bool heun_fused_preferred(Ctx& c) {
  if (c.N <= 1500000) return false;
  const FusedPlan* pl = fused_plan(c);
  return pl && pl->CX >= 8;
}

namespace {

bool build_plan(Ctx& c, FusedPlan& pl) {
  if (!heun_fused_supported(c)) return false;
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const int ny = c.d.ny, nz = c.d.nz, nx = c.d.nx;
  int smem_sm = 0, smem_cta = 0;
  cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, c.device);
  cudaDeviceGetAttribute(&smem_cta, cudaDevAttrMaxSharedMemoryPerBlockOptin, c.device);

  // Strip width: every multiple of 4 up to 64 sites; a plan is scored by the share of predictor work that is useful
  // (ragged last strip, idle lanes of the last main warp, the recomputed halo columns), with a preference for
  // 8 groups per row (a quarter-warp then reads one contiguous 128-byte row segment: conflict-free 128-bit loads)
  // and for two resident CTAs per SM (one computes while the other waits at its barrier).
  const char* force = std::getenv("ASD_FUSED_BY");          // tuning override (strip width in sites)
  const int force_by = force ? std::atoi(force) : 0;
  struct Cand { int by, shape, ctas; double score; } best{0, 0, 0, -1.0};
  for (int by = 4; by <= 64; by += 4) {
    if (force_by && by != force_by) continue;
    if (by > ny && by != (ny + 3) / 4 * 4) continue;
    const int ns = (ny + by - 1) / by, tasks = nz * (by / 4);
    const int n_main = round_up32(tasks), n_halo = round_up32(nz);
    uint32_t sp;
    const uint32_t smem = plan_smem(nz, by, sp);
    if ((int)smem > smem_cta) continue;
    for (int sh = 0; sh < kNumShapes; ++sh) {
      if (n_main + n_halo > kShapes[sh].nt) continue;
      int ctas = smem_sm / (int)(smem + 1024);
      if (ctas > kShapes[sh].minb) ctas = kShapes[sh].minb;
      if (ctas < 1) continue;
      const double useful = ((double)ny / (ns * by)) * ((double)tasks / n_main) * ((double)by / (by + 2.6));
      const double score = useful * (by == 32 ? 1.0 : 0.92) * (ctas >= 2 ? 1.0 : 0.85);
      if (score > best.score) best = Cand{by, sh, ctas, score};
      break;                                                // smallest shape that holds the tasks
    }
  }
  if (best.score < 0.0) return false;
  pl.BY = best.by; pl.G = best.by / 4; pl.nstrips = (ny + best.by - 1) / best.by;
  pl.n_main = round_up32(nz * pl.G);
  pl.threads = pl.n_main + round_up32(nz);
  pl.smem_bytes = plan_smem(nz, pl.BY, pl.slot_pitch);
  pl.kern = kernel_for(c.d.lattice, best.shape, nz, pl.BY);
  pl.kern_mm = kernel_for(c.d.lattice, best.shape, nz, pl.BY, true);
  if (pl.kern_mm && cudaFuncSetAttribute((const void*)pl.kern_mm, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)pl.smem_bytes) != cudaSuccess) {
    cudaGetLastError();
    pl.kern_mm = nullptr;
  }
  pl.kern_dm = kernel_for(c.d.lattice, best.shape, nz, pl.BY, false, true);
  {
    // Eq. (6) epilogue: [2][3][y-cells a strip can overlap][cell layers] int32 behind the field box, if that keeps the
    // CTAs per SM (else the cell sums come from coarse_grain_ydft as before)
    const int my = c.d.macro[1] > 0 ? c.d.macro[1] : 1, mz = c.d.macro[2] > 0 ? c.d.macro[2] : 1;
    pl.dm_ncyl = (uint32_t)((pl.BY - 1) / my + 2);
    const uint32_t acc_bytes = (uint32_t)align_up((size_t)2 * 3 * pl.dm_ncyl * ((nz + mz - 1) / mz) * 4, 128);
    const uint32_t with_acc = pl.smem_bytes + acc_bytes;
    pl.smem_bytes_dm = ((int)with_acc <= smem_cta && smem_sm / (int)(with_acc + 1024) >= std::min(best.ctas, smem_sm / (int)(pl.smem_bytes + 1024)))
                           ? with_acc : 0u;
  }
  if (pl.kern_dm && cudaFuncSetAttribute((const void*)pl.kern_dm, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)std::max(pl.smem_bytes, pl.smem_bytes_dm)) != cudaSuccess) {
    cudaGetLastError();
    pl.kern_dm = nullptr;
  }
  pl.kern_dm_mm = kernel_for(c.d.lattice, best.shape, nz, pl.BY, true, true);
  if (pl.kern_dm_mm && cudaFuncSetAttribute((const void*)pl.kern_dm_mm, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)std::max(pl.smem_bytes, pl.smem_bytes_dm)) != cudaSuccess) {
    cudaGetLastError();
    pl.kern_dm_mm = nullptr;
  }
  int bps = 0;
  if (cudaFuncSetAttribute((const void*)pl.kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem_bytes) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, (const void*)pl.kern, pl.threads, pl.smem_bytes) != cudaSuccess ||
      bps < 1) {
    cudaGetLastError();
    return false;
  }
  pl.ctas_per_sm = bps;
  // one wave: as many x-chunks as there are CTA slots for each strip, but chunks of at least 4 planes (every chunk
  // recomputes the predictor of 2 extra planes)
  int nchunks = (c.sm_count * bps) / pl.nstrips;
  if (nchunks > nx / 4) nchunks = nx / 4;
  if (nchunks < 1) nchunks = 1;
  const char* fc = std::getenv("ASD_FUSED_CHUNKS");         // tuning override
  if (fc && std::atoi(fc) > 0) nchunks = std::min(std::atoi(fc), nx);
  pl.CX = (nx + nchunks - 1) / nchunks;
  pl.nchunks = (nx + pl.CX - 1) / pl.CX;

  // The 13 per-site arrays as one 4-D tensor (y, z-row, x-plane, array); origin = site (0,0,0) of array 0.
  const cuuint64_t dims[4] = {(cuuint64_t)ny, (cuuint64_t)nz, (cuuint64_t)nx, (cuuint64_t)AR_COUNT};
  const cuuint64_t strides[3] = {(cuuint64_t)c.nyp * 4, (cuuint64_t)nz * c.nyp * 4, (cuuint64_t)c.as * 4};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const cuuint32_t box[4] = {(cuuint32_t)(pl.BY + 8), (cuuint32_t)(nz + 2), 1u, 3u};
  const cuuint32_t boxF[4] = {(cuuint32_t)pl.BY, (cuuint32_t)nz, 1u, 4u};     // sigma, Bx, By, Bz of one strip plane
  return enc(&pl.mapS, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)(c.arrays + c.lead), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS &&
         enc(&pl.mapF, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)(c.arrays + c.lead), dims, strides, boxF, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

bool heun_fused_takes_mm(Ctx& c) { const FusedPlan* pl = fused_plan(c); return pl && pl->kern_mm; }
bool heun_fused_takes_demag(Ctx& c, bool with_edge_field) {
  const FusedPlan* pl = fused_plan(c);
  return pl && (with_edge_field ? pl->kern_dm_mm : pl->kern_dm);
}

FusedPlan* fused_plan(Ctx& c) {
  if (!c.fused_plan_tried) {
    c.fused_plan_tried = true;
    FusedPlan* pl = new FusedPlan();
    if (build_plan(c, *pl)) c.fused_plan = pl;
    else delete pl;
  }
  return c.fused_plan;
}

void fused_plan_free(Ctx& c) {
  delete c.fused_plan;
  c.fused_plan = nullptr;
}

// One Heun step = one launch; the result lands in the scratch spin buffer, which then becomes S.
asd_status launch_heun_fused(Ctx& c, StageParams& p) {
  FusedPlan* pl = fused_plan(c);
  if (!pl) return ASD_EUNSUPPORTED;
  FusedParams f;
  f.arrays = c.arrays; f.arrays_w = c.arrays; f.as = (uint32_t)c.as;
  f.aIn = c.aS; f.oOut = (uint32_t)c.aSt * f.as;
  f.oSigma = AR_SIGMA * f.as; f.oB = AR_B * f.as;
  f.col = p.col; f.grain = p.grain;
  f.nx = c.d.nx; f.ny = c.d.ny; f.nz = c.d.nz; f.nyp = c.nyp; f.lead = c.lead;
  f.BY = pl->BY; f.G = pl->G; f.nstrips = pl->nstrips; f.CX = pl->CX; f.n_main = pl->n_main;
  f.slot_pitch = pl->slot_pitch;
  f.ngdt = -p.gdt;
  f.j1s = f.ngdt * p.jx[0]; f.j2s = f.ngdt * p.jx[1]; f.j3s = f.ngdt * p.jx[2];
  f.lambda = p.lambda; f.scale = p.scale;
  f.n_lo = p.n_lo; f.n_hi = p.n_hi; f.dyn = p.dyn; f.g0 = p.g0; f.key = p.key;
  f.edgeB = p.edgeB;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(pl->nstrips * pl->nchunks)); cfg.blockDim = dim3((unsigned)pl->threads);
  cfg.dynamicSmemBytes = pl->smem_bytes; cfg.stream = c.launch_stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  f.dm = p.dm; f.dm_my = (uint32_t)c.d.macro[1];
  const FusedKernel kern = f.dm.B ? (f.edgeB ? pl->kern_dm_mm : pl->kern_dm) : (f.edgeB ? pl->kern_mm : pl->kern);
  if (!kern || (f.dm.B && c.demag_every < 1)) return ASD_EUNSUPPORTED;
  // held-field scheme: the field of S is refreshed before the step when the cadence says so, then serves both stages
  // (from the cell sums the previous fused step left behind, when it did: demag_acc_arm below)
  if (f.dm.B && (c.demag_refresh & 1)) { const asd_status st = launch_demag(c, c.aS, true); if (st != ASD_OK) return st; }
  f.dm_acc = nullptr; f.dm_mx = (uint32_t)c.d.macro[0]; f.dm_ncyl = pl->dm_ncyl; f.dm_fx = 0.0f;
  if (f.dm.B && pl->smem_bytes_dm && c.demag_age % c.demag_every == 0) {
    // the NEXT step refreshes the held field from the spins this step writes: Eq. (6) rides with the corrector
    f.dm_acc = demag_acc_arm(c, f.dm_fx);
    if (f.dm_acc) cfg.dynamicSmemBytes = pl->smem_bytes_dm;
  }
  cudaLaunchKernelEx(&cfg, kern, pl->mapS, pl->mapF, f);
  ASD_LAUNCH_CHECK(c, "heun step (fused)");
  const int t = c.aS; c.aS = c.aSt; c.aSt = t;
  return ASD_OK;
}

}  // namespace asd
