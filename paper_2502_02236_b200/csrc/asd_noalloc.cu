// asd_noalloc.cu -- asd_spin_sum_noalloc: the window-magnetisation reduction (Eq. (6) with V = the arrays given)
// for callers that may not allocate: code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The two-stage deterministic reduction of asd_reduce.cu needs a table of per-block partial sums.  There it lives in the
// context's caller-owned workspace; here it is a file-scope array in device memory, so the entry point needs no context,
// no workspace and no allocation of any kind (no cudaMalloc / cudaFree / cudaMallocHost, no allocating library routine).
//   * Cost: kScratchBytes = 64 KB of device memory on every GPU that loads libasd.so, held until the process exits.
//   * Limit: ASD_NOALLOC_MAX_COUNT = 8 388 608 floats per component (one partial row per 4096 elements, 2048 rows);
//     larger counts are rejected with ASD_EINVAL.  cfg4's whole padded window (5.33 M) fits.
//   * The array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to start at
//     zero: a call writes rows 0 .. nb-1 in its first kernel and reads exactly those rows in its second, so stale rows of
//     a longer earlier call are never read.  Calls that OVERLAP on the GPU (two streams, two host threads, two processes'
//     worth of streams in one process) race on it: serialise them (one stream, or events between streams).
//
// In host code the array's name is a host-side stand-in, not a device address; the address the kernels get is taken once
// per device, with that device current, by cudaGetSymbolAddress (scratch_for_current_device).
#include <mutex>

#include "asd_internal.cuh"

namespace asd {

void set_static_error(const char* msg);   // asd_api.cu: what asd_last_error(NULL) returns (thread-local)

namespace {

constexpr int kRowElems = 4096;                       // elements of each component summed by one block
constexpr int kMaxRows = 2048;
constexpr size_t kMaxCount = (size_t)kRowElems * kMaxRows;          // = ASD_NOALLOC_MAX_COUNT (include/asd.h)
constexpr size_t kScratchBytes = (size_t)kMaxRows * 4 * sizeof(double);
static_assert(kMaxCount == (size_t)ASD_NOALLOC_MAX_COUNT, "include/asd.h states the limit");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
double* g_scratch_ptr[kMaxDevices] = {};              // device address of g_noalloc_scratch, per device ordinal
std::mutex g_scratch_mu;

// Device address of the scratch array on the CURRENT device (looked up once per device).  nullptr + message on failure.
double* scratch_for_current_device() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
    cudaGetLastError();
    set_static_error("asd_spin_sum_noalloc: no current CUDA device (libasd has no CPU path)");
    return nullptr;
  }
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      set_static_error("asd_spin_sum_noalloc: cudaGetSymbolAddress of the static scratch array failed");
      return nullptr;
    }
    g_scratch_ptr[dev] = static_cast<double*>(p);
  }
  return g_scratch_ptr[dev];
}

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
  return v;
}

// Stage 1: block b sums elements b*4096 .. b*4096+4095 of the three components and counts the sites that hold a spin
// (|S|^2 > 1/4: a magnetic site has |S| = 1, a vacant site or a pad float exact zeros).  Fixed partition, fixed order.
__global__ void __launch_bounds__(256) spin_sum_partial(const float* __restrict__ sx, const float* __restrict__ sy,
                                                        const float* __restrict__ sz, size_t count,
                                                        double* __restrict__ rows) {
  __shared__ double sm[4][8];
  const size_t lo = (size_t)blockIdx.x * kRowElems;
  const size_t hi = lo + kRowElems < count ? lo + kRowElems : count;
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  for (size_t l = lo + threadIdx.x; l < hi; l += blockDim.x) {
    const float x = sx[l], y = sy[l], z = sz[l];
    a0 += x; a1 += y; a2 += z;
    a3 += (x * x + y * y + z * z > 0.25f) ? 1.0 : 0.0;
  }
  a0 = warp_sum_d(a0); a1 = warp_sum_d(a1); a2 = warp_sum_d(a2); a3 = warp_sum_d(a3);
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) { sm[0][w] = a0; sm[1][w] = a1; sm[2][w] = a2; sm[3][w] = a3; }
  __syncthreads();
  if (threadIdx.x < 4) {
    double s = 0.0;
    for (int q = 0; q < 8; ++q) s += sm[threadIdx.x][q];
    rows[4 * (size_t)blockIdx.x + threadIdx.x] = s;
  }
}

// Stage 2: one warp per output sums rows 0 .. nb-1 in a fixed order.
__global__ void __launch_bounds__(128) spin_sum_final(const double* __restrict__ rows, int nb, double* __restrict__ out4) {
  const int comp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double s = 0.0;
  for (int b = lane; b < nb; b += 32) s += rows[4 * b + comp];
  s = warp_sum_d(s);
  if (lane == 0) out4[comp] = s;
}

}  // namespace

}  // namespace asd

extern "C" ASD_API asd_status asd_spin_sum_noalloc(const float* d_sx, const float* d_sy, const float* d_sz, size_t count,
                                                   double* d_out4, void* cuda_stream) {
  using namespace asd;
  if (!d_sx || !d_sy || !d_sz || !d_out4) { set_static_error("asd_spin_sum_noalloc: NULL pointer"); return ASD_EINVAL; }
  if (count == 0) { set_static_error("asd_spin_sum_noalloc: count is 0"); return ASD_EINVAL; }
  if (count > kMaxCount) {
    set_static_error("asd_spin_sum_noalloc: count exceeds ASD_NOALLOC_MAX_COUNT = 8388608 floats per component "
                     "(the static 64 KB scratch array holds one partial row per 4096); use asd_magnetisation_planes");
    return ASD_EINVAL;
  }
  double* rows = scratch_for_current_device();
  if (!rows) return ASD_ECUDA;
  const int nb = (int)((count + kRowElems - 1) / kRowElems);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  spin_sum_partial<<<nb, 256, 0, st>>>(d_sx, d_sy, d_sz, count, rows);
  spin_sum_final<<<1, 128, 0, st>>>(rows, nb, d_out4);
  if (cudaGetLastError() != cudaSuccess) { set_static_error("asd_spin_sum_noalloc: kernel launch failed"); return ASD_ECUDA; }
  return ASD_OK;
}
