// asd_graph.cu -- asd_step_heun(n) as CUDA-graph replays (the Blackwell playbook's remedy for launch-bound loops).
//
// A small lattice finishes a stage kernel in a few microseconds, less than it costs to launch it; a batch of k Heun
// steps is therefore recorded once as a graph of 2k kernel nodes and replayed.  The two values that differ from one
// replay to the next -- the step index (the Philox counter) and the head-field scale -- do not live in the frozen
// kernel parameters: the kernels read them from a DynState in device memory (asd_internal.cuh), which one 1-thread
// kernel updates in stream order before each replay.  Everything else a stage kernel is told (window origin, which
// buffer holds S, the kernel variant) changes only on a window shift or an asd_set_kernel call, and those drop the
// cache.  Graphs are recorded on an internal stream (the caller's may be the legacy default stream, which cannot be
// captured) and launched on the caller's.  Results are bit-identical to plain launches: same kernels, same order.
#include <cstring>
#include <vector>

#include "asd_internal.cuh"

namespace asd {

struct GraphCache {
  struct Entry { int64_t n; cudaGraphExec_t exec; };
  std::vector<Entry> entries;
};

namespace {

constexpr int64_t kBatch = 64;                 // Heun steps per recorded graph (128 kernel nodes)
constexpr int64_t kAutoMaxSites = 1 << 18;     // ASD_GRAPH_AUTO: lattices whose stage kernel is shorter than a launch

__global__ void set_dyn_kernel(DynState* d, uint32_t n_lo, uint32_t n_hi, float scale) {
  d->n_lo = n_lo; d->n_hi = n_hi; d->scale = scale; d->pad = 0u;
}

cudaGraphExec_t record(Ctx& c, int64_t n) {
  if (!c.cap_stream && cudaStreamCreateWithFlags(&c.cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  if (cudaStreamBeginCapture(c.cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  const int64_t launches_before = c.launches;
  const bool failed_before = c.cuda_failed;
  char err_before[sizeof(c.err)];
  std::memcpy(err_before, c.err, sizeof(c.err));
  c.launch_stream = c.cap_stream;
  const asd_status st = launch_heun_direct(c, n, dyn_state(c));
  c.launch_stream = c.stream;
  c.launches = launches_before;                // recording is not launching
  if (st != ASD_OK) {                          // a launch refused during capture is not a sticky device error:
    c.cuda_failed = failed_before;             // the caller falls back to plain launches
    std::memcpy(c.err, err_before, sizeof(c.err));
  }
  cudaGraph_t g = nullptr;
  const cudaError_t e = cudaStreamEndCapture(c.cap_stream, &g);
  if (st != ASD_OK || e != cudaSuccess || !g) {
    if (g) cudaGraphDestroy(g);
    cudaGetLastError();
    return nullptr;
  }
  cudaGraphExec_t exec = nullptr;
  if (cudaGraphInstantiate(&exec, g, 0) != cudaSuccess) { exec = nullptr; cudaGetLastError(); }
  cudaGraphDestroy(g);
  return exec;
}

cudaGraphExec_t lookup(Ctx& c, int64_t n) {
  if (!c.graphs) c.graphs = new GraphCache();
  for (auto& en : c.graphs->entries) if (en.n == n) return en.exec;
  cudaGraphExec_t exec = record(c, n);
  if (exec) c.graphs->entries.push_back({n, exec});
  return exec;
}

}  // namespace

DynState* dyn_state(const Ctx& c) { return reinterpret_cast<DynState*>(c.flags + 4); }

void graphs_invalidate(Ctx& c) {
  if (!c.graphs) return;
  for (auto& en : c.graphs->entries) cudaGraphExecDestroy(en.exec);
  c.graphs->entries.clear();
}

void graphs_free(Ctx& c) {
  graphs_invalidate(c);
  delete c.graphs;
  c.graphs = nullptr;
  if (c.cap_stream) { cudaStreamDestroy(c.cap_stream); c.cap_stream = nullptr; }
}

asd_status launch_heun(Ctx& c, int64_t n) {
  c.launch_stream = c.stream;
  const bool use = !c.demag && !edge_field_on(c) &&         // the demag pipeline and the mesh steps are launched plainly
                   c.kernel_variant != ASD_KERNEL_FUSED &&   // the fused step swaps the spin buffers every step
                   c.kernel_variant != ASD_KERNEL_PERSISTENT &&
                   !(c.kernel_variant == ASD_KERNEL_AUTO && heun_persist_preferred(c)) &&   // one launch already
                   (c.graph_mode == ASD_GRAPH_ON || (c.graph_mode == ASD_GRAPH_AUTO && c.N <= kAutoMaxSites));
  while (use && n >= 2) {
    const int64_t k = n < kBatch ? n : kBatch;
    cudaGraphExec_t exec = lookup(c, k);
    if (!exec) break;                          // cannot record here: fall through to plain launches
    set_dyn_kernel<<<1, 1, 0, c.stream>>>(dyn_state(c), (uint32_t)((uint64_t)c.step & 0xFFFFFFFFull),
                                          (uint32_t)((uint64_t)c.step >> 32), c.scale);
    ASD_LAUNCH_CHECK(c, "set_dyn");
    ASD_CUDA_TRY(c, cudaGraphLaunch(exec, c.stream));
    c.launches += 2 * k;
    c.step += k;
    n -= k;
  }
  return n > 0 ? launch_heun_direct(c, n, nullptr) : ASD_OK;
}

}  // namespace asd
