// asd_heun_ell.cu -- the hot path for a general ELL neighbour table with per-pair J (BASELINE north_star: "the L1_0 path
// uses an ELL neighbour table with per-pair J"): one fused kernel per stochastic-Heun stage.
//
//   B_ex,i = sum_s (J_is / mu_s) X_{n(i,s)},   s = 0 .. W-1,   n(i,s) = -1: no neighbour in that slot
//
// The table is slot-major (idx int32[W][N], J/mu_s fp32[W][N], entries = padded element offsets), so with ONE site per
// thread every table read is a coalesced 128-byte sweep per warp and every neighbour gather of adjacent sites lands on
// adjacent (or the same few) cache lines.  All slots of a chunk are loaded before any is used (memory-level parallelism
// without a dependent chain per slot); an empty slot is stored at set-up as (the site itself, J = 0), so the kernel has
// neither a test nor a select per slot.  The table is a pure stream: a bulk L2 prefetch runs a third of a wave ahead
// exactly as in the film kernel, and the kernels are launched with programmatic dependent launch.
//
// Bytes per site per stage that must come from / go to HBM: 52 + 8 W: 132 for the 10-neighbour L1_0
// shells.  Boundaries, vacancies, grain decoupling and periodic wraps all live in the table; the kernel knows none of it.
#include <type_traits>

#include "asd_internal.cuh"
#include "asd_site.cuh"

namespace asd {

namespace {

constexpr int kEllThreads = 256;
constexpr int kEllChunk = 5;                 // slots loaded together (W = 10: two chunks).  Measured on cfg4 (us per stage):
                                             // 5 x 256 threads x 4 CTAs/SM 151.2; 10 x 256 x 4 153.3; 5 x 128 x 8 156.1; 5 x 256 x 6 156.4
constexpr uint32_t kEllPrefetchAhead = 148;  // CTAs: a third of a wave, as in the film kernel

struct EllParams {
  const float* arrays;
  float* arrays_w;
  uint32_t as;
  uint32_t oX, oA, oOut, oOutA, oSigma, oB;
  const int32_t* idx;              // [W][N] padded element offsets (an empty slot: the site itself, with J = 0)
  const float* Jt;                 // [W][N] J / mu_s, Tesla
  int32_t W;
  uint32_t N, ny, nyp, lead, nz;
  uint32_t m_ny, s_ny, m_nz, s_nz; // multiply-high constants: l / ny and r / nz
  const uint32_t* col;             // column table at the window origin (grain id + 1 in the low 16 bits)
  const float4* grain;             // (e_x, e_y, e_z, 2 k_u/mu_s) per grain id + 1
  float gdt, lambda, scale;
  uint32_t n_lo, n_hi;
  const DynState* dyn;
  uint64_t g0;
  PhiloxKey key;
};

// base + 4 * idx as ONE widening multiply-add (the compiler's default for pointer + zero-extended index is an LEA pair)
template <class T>
__device__ __forceinline__ const T* at32(const T* base, uint32_t idx) {
  uint64_t a;
  asm("mad.wide.u32 %0, %1, 4, %2;" : "=l"(a) : "r"(idx), "l"(base));
  return reinterpret_cast<const T*>(a);
}

// WT = table width known at compile time (6: simple cubic, 10: the L1_0 shells), or 0 = read it from the parameters.
template <int STAGE, int WT>
__global__ void __launch_bounds__(kEllThreads, 4) heun_stage_ell(const EllParams p) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int W = WT > 0 ? WT : p.W;
  // ---- L2 prefetch of the streams of the CTA that runs kEllPrefetchAhead blocks later: W index rows, W J rows ----
  {
    const uint32_t lb = (blockIdx.x + kEllPrefetchAhead) * (uint32_t)kEllThreads;
    if (threadIdx.x < 2u * (uint32_t)W && lb < p.N) {
      const uint32_t s = threadIdx.x >> 1;
      const void* src = (threadIdx.x & 1u) ? (const void*)(p.Jt + (size_t)s * p.N + lb) : (const void*)(p.idx + (size_t)s * p.N + lb);
      const uint32_t room = p.N - lb;
      const uint32_t bytes = ((room < (uint32_t)kEllThreads ? room : (uint32_t)kEllThreads) * 4u) & ~15u;
      if (bytes && (((uintptr_t)src) & 15u) == 0u)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
    }
  }
  const uint32_t l = blockIdx.x * (uint32_t)kEllThreads + threadIdx.x;      // dense window-local site
  if (l >= p.N) return;
  const uint32_t r = div_u31(l, p.m_ny, p.s_ny);                            // row (i * nz + k)
  const uint32_t j = l - r * p.ny;
  const uint32_t i = div_u31(r, p.m_nz, p.s_nz);
  const uint32_t e = p.lead + r * p.nyp + j;                                // padded element of the site
  const uint32_t gid = __ldg(p.col + (i * p.ny + j)) & 0xFFFFu;             // read-only table: before the wait
  const float4 gp = __ldg(p.grain + gid);
  asm volatile("griddepcontrol.wait;" ::: "memory");

  // component bases of the configuration read through the table, and the thread's place in each stream
  const float* __restrict__ Xc0 = p.arrays + p.oX;
  const float* __restrict__ Xc1 = Xc0 + p.as;
  const float* __restrict__ Xc2 = Xc1 + p.as;
  const float* __restrict__ own = p.arrays + e;

  // ---- own spin and streamed inputs ----
  const float X0 = __ldg(Xc0 + e), X1 = __ldg(Xc1 + e), X2 = __ldg(Xc2 + e);
  const float sg = __ldg(own + p.oSigma);
  const float Bap[3] = {__ldg(own + p.oB), __ldg(own + (p.oB + p.as)), __ldg(own + (p.oB + 2u * p.as))};
  float Ai[3] = {0.0f, 0.0f, 0.0f};
  if (STAGE == 1) {
#pragma unroll
    for (int c = 0; c < 3; ++c) Ai[c] = __ldg(own + (p.oA + (uint32_t)c * p.as));
  }

  // ---- exchange field: chunks of kEllChunk slots, table first, then the gathers, then the sums.  Empty slots were
  // stored at set-up as (the site itself, J = 0): no test, no select. ----
  float Be[3] = {0.0f, 0.0f, 0.0f};
  uint32_t q = l;                                                // element offset of (slot, site) in the table: s * N + l
  auto chunk = [&](auto count) {
    constexpr int C = decltype(count)::value;
    uint32_t n[C];
    float Jt[C];
#pragma unroll
    for (int u = 0; u < C; ++u) { n[u] = (uint32_t)__ldg(at32(p.idx, q)); Jt[u] = __ldg(at32(p.Jt, q)); q += p.N; }
    float nb[C][3];
#pragma unroll
    for (int u = 0; u < C; ++u) { nb[u][0] = __ldg(at32(Xc0, n[u])); nb[u][1] = __ldg(at32(Xc1, n[u])); nb[u][2] = __ldg(at32(Xc2, n[u])); }
#pragma unroll
    for (int u = 0; u < C; ++u)
#pragma unroll
      for (int c = 0; c < 3; ++c) Be[c] = fmaf(Jt[u], nb[u][c], Be[c]);
  };
  if (WT > 0) {
#pragma unroll
    for (int s0 = 0; s0 + kEllChunk <= WT; s0 += kEllChunk) chunk(std::integral_constant<int, kEllChunk>{});
#pragma unroll
    for (int s0 = WT - WT % kEllChunk; s0 < WT; ++s0) chunk(std::integral_constant<int, 1>{});
  } else {
    int s0 = 0;
    for (; s0 + kEllChunk <= W; s0 += kEllChunk) chunk(std::integral_constant<int, kEllChunk>{});
    for (; s0 < W; ++s0) chunk(std::integral_constant<int, 1>{});
  }

  // ---- noise, torque, update, renormalise ----
  uint32_t n_lo = p.n_lo, n_hi = p.n_hi; float scale = p.scale;
  resolve_dyn(p.dyn, n_lo, n_hi, scale);
  const SiteConst sc{p.gdt, p.lambda, scale};
  uint32_t rnd[4];
  philox_site(p.key, n_lo, n_hi, p.g0 + (uint64_t)l, 0u, rnd);
  float xi[3];
  normals3(rnd, xi);
  const float Xs[3] = {X0, X1, X2};
  float ov[3], oAv[3];
  site_update<STAGE>(sc, Xs, Be, gp, Bap, sg, xi, Ai, ov, oAv);
  float* __restrict__ out = p.arrays_w + e;
#pragma unroll
  for (int c = 0; c < 3; ++c) out[p.oOut + (uint32_t)c * p.as] = ov[c];
  if (STAGE == 0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) out[p.oOutA + (uint32_t)c * p.as] = oAv[c];
  }
}

template <int WT>
void launch_ell_pair(Ctx& c, EllParams& f, unsigned blocks, bool pdl) {
  const uint32_t as = f.as;
  f.oX = (uint32_t)c.aS * as; f.oOut = (uint32_t)c.aSt * as; f.oOutA = AR_A * as; f.oA = AR_A * as;
  launch_pdl(heun_stage_ell<0, WT>, blocks, kEllThreads, c.launch_stream, f, pdl);
  c.launches += 1;
  f.oX = (uint32_t)c.aSt * as; f.oOut = (uint32_t)c.aS * as;
  launch_pdl(heun_stage_ell<1, WT>, blocks, kEllThreads, c.launch_stream, f, pdl);
  c.launches += 1;
}

}  // namespace

// The dedicated ELL kernel needs 32-bit element offsets and dense site ids; everything else lives in the table.
bool heun_ell_supported(const Ctx& c) {
  return c.d.ell_width > 0 && (int64_t)AR_COUNT * c.as < (1ll << 31) && c.N * (int64_t)c.d.ell_width < (1ll << 32) &&
         c.d.track_nx * (int64_t)c.d.ny < (1ll << 30);
}

asd_status launch_heun_ell(Ctx& c, StageParams& p) {
  EllParams f;
  f.arrays = c.arrays; f.arrays_w = c.arrays; f.as = (uint32_t)c.as;
  f.oSigma = AR_SIGMA * f.as; f.oB = AR_B * f.as;
  f.idx = c.ell_idx; f.Jt = c.ell_J; f.W = c.d.ell_width;
  f.N = (uint32_t)c.N; f.ny = (uint32_t)c.d.ny; f.nyp = (uint32_t)c.nyp; f.lead = (uint32_t)c.lead; f.nz = (uint32_t)c.d.nz;
  magic_u31(f.ny, f.m_ny, f.s_ny);
  magic_u31(f.nz, f.m_nz, f.s_nz);
  f.col = p.col; f.grain = p.grain;
  f.gdt = p.gdt; f.lambda = p.lambda; f.scale = p.scale;
  f.n_lo = p.n_lo; f.n_hi = p.n_hi; f.dyn = p.dyn; f.g0 = p.g0; f.key = p.key;
  const unsigned blocks = (unsigned)((c.N + kEllThreads - 1) / kEllThreads);
  const bool pdl = c.launch_stream == c.stream;
  if (f.W == 10) launch_ell_pair<10>(c, f, blocks, pdl);
  else if (f.W == 6) launch_ell_pair<6>(c, f, blocks, pdl);
  else launch_ell_pair<0>(c, f, blocks, pdl);
  const cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) return fail_cuda(c, err, "heun stage (ell)");
  return ASD_OK;
}

}  // namespace asd
