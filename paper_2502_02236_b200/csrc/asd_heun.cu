// asd_heun.cu -- the hot path, general variant: one fused kernel per stochastic-Heun stage.
//
//   predictor  k1 = f(S, B(S));   S~ = normalise(S + dt k1);   A = S + dt/2 k1
//   corrector  k2 = f(S~, B(S~)); S  = normalise(A + dt/2 k2)          (same xi_i in both stages)
//
// Storing A (12 B/site) instead of k1 lets the corrector run without re-reading S or recomputing k1:
// 52 B (predictor) + 52 B (corrector) = 104 B per site per Heun step.
//
// This file holds the GENERAL kernel: any periodic flags, grains that touch (per-bond masks from the column
// table), any ny (scalar path when ny % 4 != 0) and the user-supplied ELL table.  The open-boundary film with
// separated grains -- every BASELINE film config -- runs the mask-free kernel of asd_heun_fast.cu instead.
// Each thread owns VEC consecutive sites of one y-row.
#include "asd_internal.cuh"
#include "asd_site.cuh"

namespace asd {

namespace {

constexpr int LAT_SC = 0, LAT_L10 = 1, LAT_ELL = 2;

template <int VEC> struct VecIO;
template <> struct VecIO<1> {
  static __device__ __forceinline__ void ld(const float* p, float v[1]) { v[0] = __ldg(p); }
  static __device__ __forceinline__ void st(float* p, const float v[1]) { p[0] = v[0]; }
};
template <> struct VecIO<4> {
  static __device__ __forceinline__ void ld(const float* p, float v[4]) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(p));
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
  static __device__ __forceinline__ void st(float* p, const float v[4]) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
  }
};

// One y-row piece extended by one site on each side:
// e[c][0] = site j0-1, e[c][1..VEC] = sites j0..j0+VEC-1, e[c][VEC+1] = site j0+VEC.
template <int VEC>
struct Row { float e[3][VEC + 2]; };

template <int VEC>
__device__ __forceinline__ void load_row(const float* X, uint32_t as, int64_t base, bool row_ok, bool need_l,
                                         bool need_r, int dl, int dr, Row<VEC>& r) {
  // base: padded element of (row, j0); dl / dr: offsets of the j0-1 / j0+VEC sites (periodic wrap folded in)
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float* Xc = X + (size_t)c * as;
    if (row_ok) VecIO<VEC>::ld(Xc + base, &r.e[c][1]);
    else {
#pragma unroll
      for (int v = 0; v < VEC; ++v) r.e[c][1 + v] = 0.0f;
    }
    r.e[c][0] = (row_ok && need_l) ? __ldg(Xc + base + dl) : 0.0f;
    r.e[c][VEC + 1] = (row_ok && need_r) ? __ldg(Xc + base + dr) : 0.0f;
  }
}

template <int VEC, int LAT, int STAGE, bool DEMAG>
__global__ void __launch_bounds__(256) heun_stage_general(const StageParams p) {
  // programmatic dependent launch (see launch_pdl): only the read-only column table is touched before the wait
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= p.nthreads) return;
  const int r = (int)(t / p.ngrp);
  const int j0 = (int)(t - (uint32_t)r * p.ngrp) * VEC;
  const int i = r / p.nz;
  const int k = r - i * p.nz;
  const int64_t e0 = (int64_t)p.lead + (int64_t)r * p.nyp + j0;          // padded element of the first own site
  const int rowp = p.nyp;
  const int64_t planep = (int64_t)p.nz * p.nyp;
  const float* X = p.arrays + (size_t)p.aX * p.as;

  uint32_t col[VEC];
#pragma unroll
  for (int v = 0; v < VEC; ++v) col[v] = __ldg(p.col + (int64_t)i * p.ny + j0 + v);
  bool any = false;
#pragma unroll
  for (int v = 0; v < VEC; ++v) any |= (col[v] & 0xFFFFu) != 0u;
  asm volatile("griddepcontrol.wait;" ::: "memory");             // the previous kernel's stores are complete and visible
  float o[3][VEC], oA[3][VEC];
  if (!any) {                                    // all vacant: keep the buffers zero there
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int v = 0; v < VEC; ++v) { o[c][v] = 0.0f; oA[c][v] = 0.0f; }
  } else {
    // window edges in x (open boundary): the column table knows only the track ends
    if (!p.pbc_x) {
#pragma unroll
      for (int v = 0; v < VEC; ++v) {
        if (i == p.nx - 1) col[v] &= ~BOND_ALL_XP;
        if (i == 0) col[v] &= ~BOND_ALL_XM;
      }
    }
    float Bex[3][VEC];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int v = 0; v < VEC; ++v) Bex[c][v] = 0.0f;

    Row<VEC> own;
    const int dl = (j0 == 0) ? (p.ny - 1) : -1;                    // j0-1 (wraps only if periodic: else bit clear)
    const int dr = (j0 + VEC == p.ny) ? (VEC - p.ny) : VEC;        // j0+VEC
    if (LAT == LAT_ELL) {
      load_row<VEC>(X, p.as, e0, true, false, false, 0, 0, own);
      const int64_t l0 = (int64_t)r * p.ny + j0;
      for (int s = 0; s < p.ell_w; ++s) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
          const int64_t q = (int64_t)s * p.N + l0 + v;
          const int32_t n = __ldg(p.ell_idx + q);          // an empty slot holds the site itself with J = 0
          const float Jt = __ldg(p.ell_J + q);
#pragma unroll
          for (int c = 0; c < 3; ++c) Bex[c][v] = fmaf(Jt, __ldg(X + (size_t)c * p.as + n), Bex[c][v]);
        }
      }
    } else {
      const bool needL = (col[0] & (BOND_YM)) != 0u, needR = (col[VEC - 1] & (BOND_YP)) != 0u;
      load_row<VEC>(X, p.as, e0, true, needL, needR, dl, dr, own);
      // y +- 1 (shell 1)
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
          const float yp = (col[v] & BOND_YP) ? own.e[c][v + 2] : 0.0f;
          const float ym = (col[v] & BOND_YM) ? own.e[c][v] : 0.0f;
          Bex[c][v] = p.jx[0] * (yp + ym);
        }
      // z +- 1 (SC: shell 1; L1_0: shell 2) -- same column, so always the same grain
      {
        const float jz = (LAT == LAT_SC) ? p.jx[0] : p.jx[1];
        const bool zp_ok = (k < p.nz - 1) || p.pbc_z, zm_ok = (k > 0) || p.pbc_z;
        const int dzp = (k == p.nz - 1) ? -(p.nz - 1) * rowp : rowp;
        const int dzm = (k == 0) ? (p.nz - 1) * rowp : -rowp;
        Row<VEC> zr;
        load_row<VEC>(X, p.as, e0 + dzp, zp_ok, false, false, 0, 0, zr);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
          for (int v = 0; v < VEC; ++v) Bex[c][v] = fmaf(jz, zr.e[c][v + 1], Bex[c][v]);
        load_row<VEC>(X, p.as, e0 + dzm, zm_ok, false, false, 0, 0, zr);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
          for (int v = 0; v < VEC; ++v) Bex[c][v] = fmaf(jz, zr.e[c][v + 1], Bex[c][v]);
      }
      // x +- 1 (shell 1) and, for L1_0, the in-plane diagonals (shell 3)
#pragma unroll
      for (int side = 0; side < 2; ++side) {
        const uint32_t bX = side == 0 ? BOND_XP : BOND_XM;
        const uint32_t bXYP = side == 0 ? BOND_XPYP : BOND_XMYP;
        const uint32_t bXYM = side == 0 ? BOND_XPYM : BOND_XMYM;
        const int64_t dx = side == 0 ? ((i == p.nx - 1) ? -(int64_t)(p.nx - 1) * planep : planep)
                                     : ((i == 0) ? (int64_t)(p.nx - 1) * planep : -planep);
        uint32_t anyb = 0u;
#pragma unroll
        for (int v = 0; v < VEC; ++v) anyb |= col[v];
        const bool row_ok = (anyb & (bX | bXYP | bXYM)) != 0u;
        const bool nl = (LAT == LAT_L10) && (col[0] & bXYM) != 0u;
        const bool nr = (LAT == LAT_L10) && (col[VEC - 1] & bXYP) != 0u;
        Row<VEC> xr;
        load_row<VEC>(X, p.as, e0 + dx, row_ok, nl, nr, dl, dr, xr);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
          for (int v = 0; v < VEC; ++v) {
            const float xs = (col[v] & bX) ? xr.e[c][v + 1] : 0.0f;
            Bex[c][v] = fmaf(p.jx[0], xs, Bex[c][v]);
            if (LAT == LAT_L10) {
              const float dp = (col[v] & bXYP) ? xr.e[c][v + 2] : 0.0f;
              const float dm = (col[v] & bXYM) ? xr.e[c][v] : 0.0f;
              Bex[c][v] = fmaf(p.jx[2], dp + dm, Bex[c][v]);
            }
          }
      }
    }

    if (p.edgeB && LAT != LAT_ELL) {                 // multiscale window: the held mesh directions beyond the x edges
#pragma unroll
      for (int side = 0; side < 2; ++side) {
        if (i != (side == 0 ? 0 : p.nx - 1)) continue;
        const float* eb = p.edgeB + (size_t)side * 3u * (size_t)planep + (size_t)k * p.nyp + j0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          float ev[VEC];
          VecIO<VEC>::ld(eb + (size_t)c * (size_t)planep, ev);
#pragma unroll
          for (int v = 0; v < VEC; ++v) Bex[c][v] += ev[v];
        }
      }
    }
    float sg[VEC], Ba[3][VEC], Ain[3][VEC];
    VecIO<VEC>::ld(p.arrays + (size_t)AR_SIGMA * p.as + e0, sg);
#pragma unroll
    for (int c = 0; c < 3; ++c) VecIO<VEC>::ld(p.arrays + (size_t)(AR_B + c) * p.as + e0, Ba[c]);
    if (STAGE == 1) {
#pragma unroll
      for (int c = 0; c < 3; ++c) VecIO<VEC>::ld(p.arrays + (size_t)(p.aA + c) * p.as + e0, Ain[c]);
    }
    const uint64_t g = p.g0 + (uint64_t)r * (uint64_t)p.ny + (uint64_t)j0;
    uint32_t n_lo = p.n_lo, n_hi = p.n_hi; float scale = p.scale;
    resolve_dyn(p.dyn, n_lo, n_hi, scale);
    const SiteConst sc{p.gdt, p.lambda, scale};
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
      const uint32_t gid = col[v] & 0xFFFFu;
      if (gid == 0u) {
        o[0][v] = o[1][v] = o[2][v] = 0.0f;
        oA[0][v] = oA[1][v] = oA[2][v] = 0.0f;
        continue;
      }
      uint32_t rnd[4];
      philox_site(p.key, n_lo, n_hi, g + v, 0u, rnd);
      float xi[3];
      normals3(rnd, xi);
      const float4 gp = __ldg(p.grain + gid);
      const float Xs[3] = {own.e[0][v + 1], own.e[1][v + 1], own.e[2][v + 1]};
      float Be[3] = {Bex[0][v], Bex[1][v], Bex[2][v]};
      if (DEMAG) {                                   // Eq. (7): the field of the site's macrocell
        float Bd[3];
        demag_at(p.dm, (uint32_t)i, (uint32_t)(j0 + v), (uint32_t)k, Bd);
        Be[0] += Bd[0]; Be[1] += Bd[1]; Be[2] += Bd[2];
      }
      const float Bap[3] = {Ba[0][v], Ba[1][v], Ba[2][v]};
      const float Ai[3] = {Ain[0][v], Ain[1][v], Ain[2][v]};
      float ov[3], oAv[3];
      site_update<STAGE>(sc, Xs, Be, gp, Bap, sg[v], xi, Ai, ov, oAv);
      o[0][v] = ov[0]; o[1][v] = ov[1]; o[2][v] = ov[2];
      if (STAGE == 0) { oA[0][v] = oAv[0]; oA[1][v] = oAv[1]; oA[2][v] = oAv[2]; }
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) VecIO<VEC>::st(p.arrays + (size_t)(p.aOut + c) * p.as + e0, o[c]);
  if (STAGE == 0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) VecIO<VEC>::st(p.arrays + (size_t)(p.aOutA + c) * p.as + e0, oA[c]);
  }
}

template <int VEC, int LAT, bool DEMAG>
asd_status launch_pair_d(Ctx& c, StageParams& p) {
  const int threads = 256;
  p.ngrp = (uint32_t)(c.d.ny / VEC);
  p.nthreads = p.nrows * p.ngrp;
  const unsigned blocks = (p.nthreads + threads - 1) / threads;
  // predictor: X = S -> out = S~, outA = A
  p.aX = c.aS; p.aOut = c.aSt; p.aOutA = AR_A; p.aA = AR_A;
  if (DEMAG && (c.demag_refresh & 1)) { const asd_status st = launch_demag(c, c.aS); if (st != ASD_OK) return st; }
  launch_pdl(heun_stage_general<VEC, LAT, 0, DEMAG>, blocks, threads, c.launch_stream, p, c.launch_stream == c.stream);
  ASD_LAUNCH_CHECK(c, "heun predictor");
  // corrector: X = S~, A -> out = S
  p.aX = c.aSt; p.aOut = c.aS;
  if (DEMAG && (c.demag_refresh & 2)) { const asd_status st = launch_demag(c, c.aSt); if (st != ASD_OK) return st; }
  launch_pdl(heun_stage_general<VEC, LAT, 1, DEMAG>, blocks, threads, c.launch_stream, p, c.launch_stream == c.stream);
  ASD_LAUNCH_CHECK(c, "heun corrector");
  return ASD_OK;
}

template <int VEC, int LAT>
asd_status launch_pair(Ctx& c, StageParams& p) {
  return p.dm.B ? launch_pair_d<VEC, LAT, true>(c, p) : launch_pair_d<VEC, LAT, false>(c, p);
}

}  // namespace

void fill_stage_params(const Ctx& c, StageParams& p) {
  p.arrays = c.arrays; p.as = (uint32_t)c.as;
  p.col = c.col_win();
  p.grain = c.grain;
  const size_t ncol = (size_t)(c.d.track_nx * c.d.ny);
  p.aniso = c.aniso + c.x0 * c.d.ny; p.aniso_stride = (uint32_t)ncol;
  p.ell_idx = c.ell_idx; p.ell_J = c.ell_J; p.ell_w = c.d.ell_width;
  p.nx = c.d.nx; p.ny = c.d.ny; p.nz = c.d.nz; p.nyp = c.nyp; p.lead = c.lead;
  p.nrows = (uint32_t)c.nrows; p.N = (uint32_t)c.N;
  p.pbc_x = c.d.pbc[0]; p.pbc_y = c.d.pbc[1]; p.pbc_z = c.d.pbc[2];
  for (int a = 0; a < 3; ++a) p.jx[a] = (float)(c.d.J[a] / c.d.mu_s);
  p.gdt = (float)(c.gamma * c.d.dt / (1.0 + c.d.lambda * c.d.lambda));
  p.lambda = (float)c.d.lambda;
  p.scale = c.scale;
  p.g0 = (uint64_t)c.x0 * (uint64_t)c.plane;
  demag_fill_params(c, p);
  p.edgeB = mm_edge_field(c);
  uint32_t k0 = (uint32_t)(c.d.seed & 0xFFFFFFFFull), k1 = (uint32_t)(c.d.seed >> 32);
  for (int r = 0; r < 10; ++r) {
    p.key.k0[r] = k0; p.key.k1[r] = k1;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
}

// n Heun steps as 2n plain launches on c.launch_stream.  dyn == nullptr: step indices come from c.step, which advances.
// dyn != nullptr (graph capture): step s of the batch carries the offset s and reads the base from *dyn; c.step is
// left to the caller.
asd_status launch_heun_direct(Ctx& c, int64_t n, const DynState* dyn) {
  StageParams p;
  fill_stage_params(c, p);
  p.dyn = dyn;
  const bool vec4 = (c.d.ny % 4 == 0);
  // with the demagnetising field on, the film kernel assumes its 4 sites span at most two macrocells (my >= 3)
  const bool fast = c.kernel_variant != ASD_KERNEL_GENERAL && heun_fast_supported(c) && !(c.demag && c.d.macro[1] < 3);
  if (c.kernel_variant == ASD_KERNEL_FAST && !fast) return ASD_EUNSUPPORTED;
  const bool staged = c.kernel_variant == ASD_KERNEL_TMA;
  if (staged && !(heun_tma_supported(c) && tma_plan(c))) return ASD_EUNSUPPORTED;
  if (c.demag && (staged || c.d.ell_width > 0)) return ASD_EUNSUPPORTED;   // demag: film and general kernels only
  if (edge_field_on(c) && (staged || dyn)) return ASD_EUNSUPPORTED;                    // multiscale: film, fused and general kernels, plain launches
  // one kernel per step: asked for, or AUTO on a film large enough to fill the machine with strip x chunk CTAs.
  // Not inside a recorded graph (the spin buffers swap roles every step) and not with the demagnetising field.
  // With the demagnetising field: only in the held-field scheme (asd_set_demag_every >= 1; the per-stage scheme needs the
  // field of S~, a global quantity, between the two stages), macrocells of >= 3 sites across.
  const bool fused_dm_ok = !c.demag || (c.demag_every >= 1 && c.d.macro[1] >= 3 && heun_fused_takes_demag(c, edge_field_on(c)));
  const bool fused = !dyn && fused_dm_ok && heun_fused_supported(c) &&
                     (c.kernel_variant == ASD_KERNEL_FUSED || (c.kernel_variant == ASD_KERNEL_AUTO && heun_fused_preferred(c))) &&
                     fused_plan(c) && (!edge_field_on(c) || heun_fused_takes_mm(c));
  if (c.kernel_variant == ASD_KERNEL_FUSED && !fused) return ASD_EUNSUPPORTED;
  // a lattice that fits one thread-block cluster's shared memory: all n steps in one launch (asd_heun_persist.cu)
  const bool persist = !dyn && heun_persist_supported(c) &&
                       (c.kernel_variant == ASD_KERNEL_PERSISTENT || (c.kernel_variant == ASD_KERNEL_AUTO && heun_persist_preferred(c)));
  if (c.kernel_variant == ASD_KERNEL_PERSISTENT && !persist) return ASD_EUNSUPPORTED;
  if (persist) return n > 0 ? launch_heun_persist(c, p, n) : ASD_OK;
  for (int64_t s = 0; s < n; ++s) {
    const uint64_t idx = dyn ? (uint64_t)s : (uint64_t)c.step;
    p.n_lo = (uint32_t)(idx & 0xFFFFFFFFull);
    p.n_hi = (uint32_t)(idx >> 32);
    if (c.mm) { const asd_status sm = mm_before_step(c); if (sm != ASD_OK) return sm; }
    if (c.demag) {
      c.demag_refresh = c.demag_every <= 0 ? 3 : (c.demag_age % c.demag_every == 0 ? 1 : 0);
      c.demag_age += 1;
    }
    if (c.demag && !fused) demag_acc_drop(c);           // cell sums a fused step left behind: of spins about to change
    asd_status st;
    if (fused) st = launch_heun_fused(c, p);
    else if (staged) st = launch_heun_tma(c, p);
    else if (fast) st = launch_heun_fast(c, p);
    else if (c.d.ell_width > 0) st = (c.kernel_variant != ASD_KERNEL_GENERAL && heun_ell_supported(c)) ? launch_heun_ell(c, p)
                                                                                                     : launch_pair<1, LAT_ELL>(c, p);
    else if (c.d.lattice == ASD_SC) st = vec4 ? launch_pair<4, LAT_SC>(c, p) : launch_pair<1, LAT_SC>(c, p);
    else st = vec4 ? launch_pair<4, LAT_L10>(c, p) : launch_pair<1, LAT_L10>(c, p);
    if (st != ASD_OK) return st;
    if (!dyn) c.step += 1;
  }
  return ASD_OK;
}

}  // namespace asd
