// asd_reduce.cu -- window and per-grain magnetisation (Eq. (6), with V = window / grain).
// Deterministic: fixed partition, fixed order, no floating-point atomics.
#include "asd_internal.cuh"

namespace asd {

namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
  return v;
}

// Stage 1: block b sums the sites b*chunk .. (b+1)*chunk-1 (vacant sites hold 0) and counts magnetic columns.
__global__ void __launch_bounds__(256) mag_partial(const float* __restrict__ sx, const float* __restrict__ sy,
                                                   const float* __restrict__ sz, const uint32_t* __restrict__ col,
                                                   int64_t N, int64_t ncol, double* __restrict__ partials) {
  __shared__ double sm[4][8];
  const int64_t chunk = (N + gridDim.x - 1) / gridDim.x;
  const int64_t lo = (int64_t)blockIdx.x * chunk, hi = min(lo + chunk, N);
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  for (int64_t l = lo + threadIdx.x; l < hi; l += blockDim.x) { a0 += sx[l]; a1 += sy[l]; a2 += sz[l]; }
  const int64_t cchunk = (ncol + gridDim.x - 1) / gridDim.x;
  const int64_t clo = (int64_t)blockIdx.x * cchunk, chi = min(clo + cchunk, ncol);
  for (int64_t t = clo + threadIdx.x; t < chi; t += blockDim.x) a3 += (col[t] & 0xFFFFu) ? 1.0 : 0.0;
  a0 = warp_sum(a0); a1 = warp_sum(a1); a2 = warp_sum(a2); a3 = warp_sum(a3);
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) { sm[0][w] = a0; sm[1][w] = a1; sm[2][w] = a2; sm[3][w] = a3; }
  __syncthreads();
  if (threadIdx.x < 4) {
    double s = 0.0;
    for (int q = 0; q < (int)(blockDim.x >> 5); ++q) s += sm[threadIdx.x][q];
    partials[4 * (int64_t)blockIdx.x + threadIdx.x] = s;
  }
}

// Stage 2: one warp per component sums the block partials in a fixed order; result in partials[0..3] of `out`.
__global__ void mag_final(const double* __restrict__ partials, int nb, double* __restrict__ out) {
  const int comp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double s = 0.0;
  for (int b = lane; b < nb; b += 32) s += partials[4 * b + comp];
  s = warp_sum(s);
  if (lane == 0) out[comp] = s;
}

// Per grain: one thread per window column sums its nz sites, then adds 32.32 fixed-point integers atomically --
// integer addition commutes, so the result does not depend on the order of the atomics.
__global__ void grain_accumulate(const float* __restrict__ sx, const float* __restrict__ sy,
                                 const float* __restrict__ sz, const uint32_t* __restrict__ col, int nx, int ny, int nz,
                                 int nyp, int lead, long long* __restrict__ acc) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (int64_t)nx * ny) return;
  const uint32_t gid = col[t] & 0xFFFFu;
  if (gid == 0u) return;
  const int i = (int)(t / ny), j = (int)(t - (int64_t)i * ny);
  long long q0 = 0, q1 = 0, q2 = 0;
  for (int k = 0; k < nz; ++k) {
    const int64_t l = lead + ((int64_t)i * nz + k) * nyp + j;
    q0 += __double2ll_rn((double)sx[l] * 4294967296.0);
    q1 += __double2ll_rn((double)sy[l] * 4294967296.0);
    q2 += __double2ll_rn((double)sz[l] * 4294967296.0);
  }
  unsigned long long* a = reinterpret_cast<unsigned long long*>(acc) + 4 * (int64_t)(gid - 1u);
  atomicAdd(a + 0, (unsigned long long)q0);
  atomicAdd(a + 1, (unsigned long long)q1);
  atomicAdd(a + 2, (unsigned long long)q2);
  atomicAdd(a + 3, (unsigned long long)nz);
}

}  // namespace

asd_status launch_magnetisation(Ctx& c, double out4[4], int32_t i0, int32_t n) {
  const int64_t planep = (int64_t)c.d.nz * c.nyp;
  const int64_t first = i0 < 0 ? 0 : (int64_t)c.lead + (int64_t)i0 * planep;       // i0 < 0: the whole padded array
  const int64_t count = i0 < 0 ? c.Np : (int64_t)n * planep;
  const int64_t ncol = i0 < 0 ? (int64_t)c.d.nx * c.d.ny : (int64_t)n * c.d.ny;
  const uint32_t* col = c.col_win() + (i0 < 0 ? 0 : (int64_t)i0 * c.d.ny);
  const int nb = (int)min((int64_t)kMaxPartialBlocks - 1, max((int64_t)1, count / 4096));
  double* final_slot = c.partials + 4 * (int64_t)(kMaxPartialBlocks - 1);
  // the padded arrays are summed whole: pads and vacant sites hold exact zeros
  const Vec3Ptr S = c.S();
  mag_partial<<<nb, 256, 0, c.stream>>>(S.x + first, S.y + first, S.z + first, col, count, ncol, c.partials);
  ASD_LAUNCH_CHECK(c, "mag_partial");
  mag_final<<<1, 128, 0, c.stream>>>(c.partials, nb, final_slot);
  ASD_LAUNCH_CHECK(c, "mag_final");
  ASD_CUDA_TRY(c, cudaMemcpyAsync(c.host_scratch, final_slot, 4 * sizeof(double), cudaMemcpyDeviceToHost, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  for (int a = 0; a < 4; ++a) out4[a] = c.host_scratch[a];
  out4[3] *= (double)c.d.nz;                     // magnetic columns -> magnetic sites
  return ASD_OK;
}

asd_status launch_grain_magnetisation(Ctx& c, double* m_host) {
  const int G = c.d.n_grains;
  ASD_CUDA_TRY(c, cudaMemsetAsync(c.grain_acc, 0, sizeof(long long) * 4 * (size_t)G, c.stream));
  const int64_t ncol = (int64_t)c.d.nx * c.d.ny;
  const Vec3Ptr S = c.S();
  grain_accumulate<<<(unsigned)((ncol + 127) / 128), 128, 0, c.stream>>>(S.x, S.y, S.z, c.col_win(), c.d.nx, c.d.ny,
                                                                        c.d.nz, c.nyp, c.lead, c.grain_acc);
  ASD_LAUNCH_CHECK(c, "grain_accumulate");
  long long* h = c.grain_scratch;                      // pinned, allocated once at create time
  ASD_CUDA_TRY(c, cudaMemcpyAsync(h, c.grain_acc, sizeof(long long) * 4 * (size_t)G, cudaMemcpyDeviceToHost, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  for (int g = 0; g < G; ++g) {
    const double cnt = (double)h[4 * g + 3];
    for (int a = 0; a < 3; ++a)
      m_host[3 * g + a] = cnt > 0.0 ? ((double)h[4 * g + a] / 4294967296.0) / cnt : 0.0;
  }
  return ASD_OK;
}

}  // namespace asd
