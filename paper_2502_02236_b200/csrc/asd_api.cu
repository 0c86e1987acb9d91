// asd_api.cu -- the C ABI of include/asd.h: argument validation, workspace layout, state, stream plumbing.
// Every arithmetic step of the method runs in the kernels of asd_heun.cu / asd_shift.cu / asd_reduce.cu /
// asd_setup.cu; this file only marshals.
#include <cmath>
#include <cstring>
#include <new>

#include "asd_internal.cuh"

namespace asd {

// message of the last failure that has no context to carry it (create, NULL ctx); per thread, not process-wide
static thread_local const char* g_static_err = "no error";
void set_static_error(const char* msg) { g_static_err = msg; }   // for entry points outside this file (asd_noalloc.cu)

bool validate_desc(const asd_lattice_desc* d, const char** why) {
  auto bad = [&](const char* m) { if (why) *why = m; return false; };
  if (!d) return bad("desc is NULL");
  if (d->lattice != ASD_SC && d->lattice != ASD_L10_FE) return bad("lattice must be ASD_SC or ASD_L10_FE");
  if (d->nx < 1 || d->ny < 1 || d->nz < 1) return bad("nx, ny, nz must be >= 1");
  if ((int64_t)d->nx * d->ny * d->nz > 2000000000LL) return bad("more than 2e9 sites");
  const int n[3] = {d->nx, d->ny, d->nz};
  for (int a = 0; a < 3; ++a) {
    if (d->pbc[a] != 0 && d->pbc[a] != 1) return bad("pbc flags must be 0 or 1");
    if (d->pbc[a] && n[a] < 3) return bad("a periodic dimension needs n >= 3");
    if (d->macro[a] < 1) return bad("macro[] must be >= 1");
    if (!std::isfinite(d->J[a])) return bad("J[] must be finite");
  }
  if (!(d->mu_s > 0.0) || !std::isfinite(d->mu_s)) return bad("mu_s must be > 0");
  if (!(d->lambda >= 0.0) || !std::isfinite(d->lambda)) return bad("lambda must be >= 0");
  if (!(d->dt > 0.0) || !std::isfinite(d->dt)) return bad("dt must be > 0");
  if (!std::isfinite(d->gamma)) return bad("gamma must be finite");
  if (d->x0 < 0 || d->track_nx < d->x0 + d->nx) return bad("track_nx must be >= x0 + nx and x0 >= 0");
  if (d->pbc[0] && (d->track_nx != d->nx || d->x0 != 0)) return bad("pbc[0] requires track_nx == nx and x0 == 0");
  if (d->track_nx * (int64_t)d->ny > 2000000000LL) return bad("grain map too large");
  if (d->n_grains < 1 || d->n_grains > 65535) return bad("n_grains must be in 1..65535");
  if (d->grain_map) {
    const int64_t n = d->track_nx * d->ny;
    for (int64_t t = 0; t < n; ++t)
      if (d->grain_map[t] < -1 || d->grain_map[t] >= d->n_grains) return bad("grain id out of range");
  }
  if (d->grain_axis) {
    for (int g = 0; g < d->n_grains; ++g) {
      const double x = d->grain_axis[3 * g], y = d->grain_axis[3 * g + 1], z = d->grain_axis[3 * g + 2];
      if (!(std::fabs(std::sqrt(x * x + y * y + z * z) - 1.0) <= 1e-4)) return bad("grain_axis must be unit vectors");
    }
  }
  if (d->grain_ku)
    for (int g = 0; g < d->n_grains; ++g)
      if (!std::isfinite(d->grain_ku[g])) return bad("grain_ku must be finite");
  if (d->ell_width < 0 || d->ell_width > 16) return bad("ell_width must be in 0..16");
  if (d->ell_width > 0 && (!d->ell_idx || !d->ell_J)) return bad("ell_width > 0 needs ell_idx and ell_J");
  return true;
}

bool compute_layout(const asd_lattice_desc& d, Layout& L) {
  L.N = (int64_t)d.nx * d.ny * d.nz;
  L.nyp = (int32_t)align_up((size_t)d.ny, 4) + 4;
  L.lead = L.nyp + 4;
  L.nrows = (int64_t)d.nx * d.nz;
  L.Np = L.lead + L.nrows * L.nyp;
  L.as = (int64_t)align_up((size_t)L.Np + 8, 64);     // +8: the last row's y+1 edge read of a redirected row stays inside
  L.ncx = (d.track_nx + d.macro[0] - 1) / d.macro[0];
  L.ncy = (d.ny + d.macro[1] - 1) / d.macro[1];
  L.ncz = (d.nz + d.macro[2] - 1) / d.macro[2];
  L.ncell = L.ncx * L.ncy * L.ncz;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes, 256); return o; };
  L.arrays = take(sizeof(float) * (size_t)L.as * AR_COUNT);
  const size_t ncol = (size_t)(d.track_nx * d.ny);
  L.col = take(sizeof(uint32_t) * ncol);
  L.gmap = take(sizeof(int32_t) * ncol);
  L.grain = take(sizeof(float4) * ((size_t)d.n_grains + 1));
  L.aniso = take(sizeof(float) * 4 * ncol + 64);
  L.flags = take(sizeof(int32_t) * 16);
  const size_t ell = (size_t)d.ell_width * (size_t)L.N;
  L.ell_idx = take(sizeof(int32_t) * ell * 2);   // slot-major table + staging for the site-major upload
  L.ell_J = take(sizeof(float) * ell * 2);
  L.init_mean = take(sizeof(float) * 3 * (size_t)L.ncell);
  L.cell_frame = take(sizeof(float) * 12 * (size_t)L.ncell);
  L.out_sum = take(sizeof(double) * 3 * (size_t)L.ncell);
  L.out_cnt = take(sizeof(long long) * (size_t)L.ncell);
  L.partials = take(sizeof(double) * 4 * kMaxPartialBlocks);
  L.grain_acc = take(sizeof(long long) * 4 * (size_t)d.n_grains);
  L.total = off;
  return true;
}

asd_status fail_cuda(Ctx& c, cudaError_t e, const char* where) {
  c.cuda_failed = true;
  std::snprintf(c.err, sizeof(c.err), "CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), where);
  return ASD_ECUDA;
}

static asd_status fail(Ctx& c, asd_status s, const char* msg) {
  std::snprintf(c.err, sizeof(c.err), "%s", msg);
  return s;
}

}  // namespace asd

using namespace asd;

#define CTX_OR_RETURN(ctx)                                         \
  if (!(ctx)) { g_static_err = "ctx is NULL"; return ASD_EINVAL; } \
  Ctx& c = (ctx)->c;                                               \
  if (c.cuda_failed) return ASD_ECUDA;

extern "C" {

size_t asd_workspace_bytes(const asd_lattice_desc* desc) {
  const char* why = nullptr;
  if (!validate_desc(desc, &why)) { g_static_err = why; return 0; }
  Layout L;
  compute_layout(*desc, L);
  return L.total;
}

asd_status asd_create_lattice(const asd_lattice_desc* desc, void* d_workspace, size_t bytes, void* cuda_stream,
                              asd_ctx** out) {
  const char* why = nullptr;
  if (!out) { g_static_err = "out is NULL"; return ASD_EINVAL; }
  *out = nullptr;
  if (!validate_desc(desc, &why)) { g_static_err = why; return ASD_EINVAL; }
  if (!d_workspace || ((uintptr_t)d_workspace & 255u)) { g_static_err = "workspace NULL or not 256-byte aligned"; return ASD_EINVAL; }
  Layout L;
  compute_layout(*desc, L);
  if (bytes < L.total) { g_static_err = "workspace too small"; return ASD_ENOMEM; }
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { g_static_err = "no CUDA device (libasd has no CPU path)"; return ASD_ECUDA; }
  asd_ctx* h = new (std::nothrow) asd_ctx();
  if (!h) { g_static_err = "out of host memory"; return ASD_ENOMEM; }
  Ctx& c = h->c;
  c.d = *desc;
  c.stream = (cudaStream_t)cuda_stream;
  c.launch_stream = c.stream;
  c.device = dev;
  cudaDeviceGetAttribute(&c.sm_count, cudaDevAttrMultiProcessorCount, dev);
  c.N = L.N; c.nyp = L.nyp; c.lead = L.lead; c.nrows = L.nrows; c.Np = L.Np; c.as = L.as;
  c.plane = desc->ny * desc->nz;
  c.gamma = desc->gamma > 0.0 ? desc->gamma : kGammaDefault;
  c.x0 = desc->x0;
  c.ncx = L.ncx; c.ncy = L.ncy; c.ncz = L.ncz; c.ncell = L.ncell;
  char* base = (char*)d_workspace;
  c.arrays = (float*)(base + L.arrays);
  c.aniso = (float*)(base + L.aniso);
  c.flags = (int32_t*)(base + L.flags);
  c.col = (uint32_t*)(base + L.col);
  c.grain_map_dev = (int32_t*)(base + L.gmap);
  c.grain = (float4*)(base + L.grain);
  c.ell_idx = desc->ell_width > 0 ? (int32_t*)(base + L.ell_idx) : nullptr;
  c.ell_J = desc->ell_width > 0 ? (float*)(base + L.ell_J) : nullptr;
  c.init_mean = (float*)(base + L.init_mean);
  c.cell_frame = (float*)(base + L.cell_frame);
  c.out_sum = (double*)(base + L.out_sum);
  c.out_cnt = (long long*)(base + L.out_cnt);
  c.partials = (double*)(base + L.partials);
  c.grain_acc = (long long*)(base + L.grain_acc);

  auto bail = [&](asd_status s) { g_static_err = "asd_create_lattice failed in CUDA set-up (see stderr)";
                                  std::fprintf(stderr, "libasd: %s\n", c.err);
                                  if (c.host_scratch) cudaFreeHost(c.host_scratch);
                                  if (c.grain_scratch) cudaFreeHost(c.grain_scratch);
                                  delete h; return s; };
#define CREATE_TRY(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { fail_cuda(c, e__, #expr); return bail(ASD_ECUDA); } } while (0)
  CREATE_TRY(cudaMallocHost(&c.host_scratch, 4 * sizeof(double)));
  CREATE_TRY(cudaMallocHost(&c.grain_scratch, sizeof(long long) * 4 * (size_t)desc->n_grains));
  CREATE_TRY(cudaMemsetAsync(d_workspace, 0, L.total, c.stream));
  const size_t ncol = (size_t)(desc->track_nx * desc->ny);
  if (desc->grain_map)
    CREATE_TRY(cudaMemcpyAsync(c.grain_map_dev, desc->grain_map, sizeof(int32_t) * ncol, cudaMemcpyHostToDevice, c.stream));
  // per-grain (e, 2 k_u / mu_s)
  {
    float4* gp = nullptr;
    CREATE_TRY(cudaMallocHost(&gp, sizeof(float4) * ((size_t)desc->n_grains + 1)));
    gp[0] = make_float4(0.f, 0.f, 1.f, 0.f);           // vacant columns: no anisotropy
    for (int g = 0; g < desc->n_grains; ++g) {
      float4 v = make_float4(0.f, 0.f, 1.f, 0.f);
      if (desc->grain_axis) { v.x = desc->grain_axis[3 * g]; v.y = desc->grain_axis[3 * g + 1]; v.z = desc->grain_axis[3 * g + 2]; }
      if (desc->grain_ku) v.w = (float)(2.0 * (double)desc->grain_ku[g] / desc->mu_s);
      gp[g + 1] = v;
    }
    cudaError_t e2 = cudaMemcpyAsync(c.grain, gp, sizeof(float4) * ((size_t)desc->n_grains + 1), cudaMemcpyHostToDevice, c.stream);
    if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(c.stream);
    cudaFreeHost(gp);
    CREATE_TRY(e2);
  }
  if (!desc->grain_map) c.grain_map_dev = nullptr;   // kernel treats NULL as "grain 0 everywhere"
  if (launch_build_columns(c) != ASD_OK) return bail(ASD_ECUDA);
  {
    int32_t touch = 1;
    CREATE_TRY(cudaMemcpyAsync(&touch, c.flags, sizeof(int32_t), cudaMemcpyDeviceToHost, c.stream));
    CREATE_TRY(cudaStreamSynchronize(c.stream));
    c.grains_touch = touch != 0;
  }
  if (desc->ell_width > 0) {
    const size_t ell = (size_t)desc->ell_width * (size_t)L.N;
    int32_t* stage_i = c.ell_idx + ell;
    float* stage_J = c.ell_J + ell;
    CREATE_TRY(cudaMemcpyAsync(stage_i, desc->ell_idx, sizeof(int32_t) * ell, cudaMemcpyHostToDevice, c.stream));
    CREATE_TRY(cudaMemcpyAsync(stage_J, desc->ell_J, sizeof(float) * ell, cudaMemcpyHostToDevice, c.stream));
    if (launch_ell_transpose(c, stage_i, stage_J) != ASD_OK) return bail(ASD_ECUDA);
  }
  if (launch_pack_spins(c, CVec3Ptr{nullptr, nullptr, nullptr}, c.S()) != ASD_OK) return bail(ASD_ECUDA);
  // track initial state: +z, m0 = 1
  {
    float* im = nullptr;
    CREATE_TRY(cudaMallocHost(&im, sizeof(float) * 3 * (size_t)L.ncell));
    for (int64_t q = 0; q < L.ncell; ++q) { im[3 * q] = 0.f; im[3 * q + 1] = 0.f; im[3 * q + 2] = 1.f; }
    cudaError_t e2 = cudaMemcpyAsync(c.init_mean, im, sizeof(float) * 3 * (size_t)L.ncell, cudaMemcpyHostToDevice, c.stream);
    if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(c.stream);
    cudaFreeHost(im);
    CREATE_TRY(e2);
  }
  if (launch_cell_frames(c) != ASD_OK) return bail(ASD_ECUDA);
  CREATE_TRY(cudaStreamSynchronize(c.stream));
#undef CREATE_TRY
  // host pointers of the description are not kept
  c.d.grain_map = nullptr; c.d.grain_ku = nullptr; c.d.grain_axis = nullptr; c.d.ell_idx = nullptr; c.d.ell_J = nullptr;
  *out = h;
  return ASD_OK;
}

asd_status asd_destroy(asd_ctx* ctx) {
  if (!ctx) return ASD_EINVAL;
  if (ctx->c.host_scratch) cudaFreeHost(ctx->c.host_scratch);
  if (ctx->c.grain_scratch) cudaFreeHost(ctx->c.grain_scratch);
  asd::tma_plan_free(ctx->c);
  asd::fused_plan_free(ctx->c);
  asd::graphs_free(ctx->c);
  if (ctx->c.copy_stream) { cudaStreamDestroy(ctx->c.copy_stream); cudaEventDestroy(ctx->c.staged_ev); cudaEventDestroy(ctx->c.consumed_ev); }
  asd::demag_free(ctx->c);
  asd::mm_free(ctx->c);
  delete ctx;
  return ASD_OK;
}

// Host uploads are staged densely in the A arrays (free between steps: A lives only from a predictor to its
// corrector, and nothing reads A's padding), then packed into the padded-row layout by a kernel.
static asd_status set_spins_impl(Ctx& c, const float* sx, const float* sy, const float* sz, bool host) {
  if (!sx || !sy || !sz) return fail(c, ASD_EINVAL, "asd_set_spins: NULL pointer");
  demag_held_invalidate(c);                             // a held demagnetising field belongs to the old spins
  mm_restart_cadence(c);                       // ... and so do the held mesh boundary data
  if (host) {
    const float* src[3] = {sx, sy, sz};
    for (int a = 0; a < 3; ++a)
      ASD_CUDA_TRY(c, cudaMemcpyAsync(c.arr(AR_A + a), src[a], sizeof(float) * (size_t)c.N, cudaMemcpyHostToDevice, c.stream));
    return launch_pack_spins(c, CVec3Ptr{c.arr(AR_A), c.arr(AR_A + 1), c.arr(AR_A + 2)}, c.S());
  }
  return launch_pack_spins(c, CVec3Ptr{sx, sy, sz}, c.S());
}

asd_status asd_set_spins(asd_ctx* ctx, const float* sx, const float* sy, const float* sz) {
  CTX_OR_RETURN(ctx);
  return set_spins_impl(c, sx, sy, sz, false);
}
asd_status asd_set_spins_host(asd_ctx* ctx, const float* sx, const float* sy, const float* sz) {
  CTX_OR_RETURN(ctx);
  return set_spins_impl(c, sx, sy, sz, true);
}

static asd_status get_spins_impl(Ctx& c, float* sx, float* sy, float* sz, bool host) {
  if (!sx || !sy || !sz) return fail(c, ASD_EINVAL, "asd_get_spins: NULL pointer");
  float* dst[3] = {sx, sy, sz};
  const Vec3Ptr S = c.S();
  const float* src[3] = {S.x, S.y, S.z};
  for (int a = 0; a < 3; ++a) {
    if (host) {
      const asd_status st = launch_unpack(c, src[a], c.arr(AR_A + a));
      if (st != ASD_OK) return st;
      ASD_CUDA_TRY(c, cudaMemcpyAsync(dst[a], c.arr(AR_A + a), sizeof(float) * (size_t)c.N, cudaMemcpyDeviceToHost, c.stream));
    } else {
      const asd_status st = launch_unpack(c, src[a], dst[a]);
      if (st != ASD_OK) return st;
    }
  }
  if (host) ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  return ASD_OK;
}
asd_status asd_get_spins(asd_ctx* ctx, float* sx, float* sy, float* sz) {
  CTX_OR_RETURN(ctx);
  return get_spins_impl(c, sx, sy, sz, false);
}
asd_status asd_get_spins_host(asd_ctx* ctx, float* sx, float* sy, float* sz) {
  CTX_OR_RETURN(ctx);
  return get_spins_impl(c, sx, sy, sz, true);
}

static asd_status set_fields_impl(Ctx& c, const float* T, const float* Bx, const float* By, const float* Bz,
                                  bool host) {
  const size_t b = sizeof(float) * (size_t)c.N;
  const float* Bsrc[3] = {Bx, By, Bz};
  for (int a = 0; a < 3; ++a) {
    if (!Bsrc[a]) continue;
    const float* dense = Bsrc[a];
    if (host) {
      ASD_CUDA_TRY(c, cudaMemcpyAsync(c.arr(AR_A + a), Bsrc[a], b, cudaMemcpyHostToDevice, c.stream));
      dense = c.arr(AR_A + a);
    }
    const asd_status st = launch_pack_field(c, dense, c.B(a));
    if (st != ASD_OK) return st;
  }
  if (T) {
    const float* dense = T;
    if (host) {
      ASD_CUDA_TRY(c, cudaMemcpyAsync(c.arr(AR_A), T, b, cudaMemcpyHostToDevice, c.stream));
      dense = c.arr(AR_A);
    }
    return launch_sigma(c, dense);
  }
  return ASD_OK;
}
asd_status asd_set_fields(asd_ctx* ctx, const float* T, const float* Bx, const float* By, const float* Bz) {
  CTX_OR_RETURN(ctx);
  return set_fields_impl(c, T, Bx, By, Bz, false);
}
asd_status asd_set_fields_host(asd_ctx* ctx, const float* T, const float* Bx, const float* By, const float* Bz) {
  CTX_OR_RETURN(ctx);
  return set_fields_impl(c, T, Bx, By, Bz, true);
}

size_t asd_staging_bytes(const asd_ctx* ctx) {
  if (!ctx) return 0;
  return 4 * align_up(sizeof(float) * (size_t)ctx->c.N, 256);
}

asd_status asd_set_staging(asd_ctx* ctx, void* d_staging, size_t bytes) {
  CTX_OR_RETURN(ctx);
  if (!d_staging || ((uintptr_t)d_staging & 255u)) return fail(c, ASD_EINVAL, "asd_set_staging: NULL or not 256-byte aligned");
  if (bytes < asd_staging_bytes(ctx)) return fail(c, ASD_ENOMEM, "asd_set_staging: buffer too small");
  if (!c.copy_stream) {
    ASD_CUDA_TRY(c, cudaStreamCreateWithFlags(&c.copy_stream, cudaStreamNonBlocking));
    ASD_CUDA_TRY(c, cudaEventCreateWithFlags(&c.staged_ev, cudaEventDisableTiming));
    ASD_CUDA_TRY(c, cudaEventCreateWithFlags(&c.consumed_ev, cudaEventDisableTiming));
  }
  c.staging = (float*)d_staging;
  c.staged_mask = 0;
  return ASD_OK;
}

asd_status asd_stage_fields_host(asd_ctx* ctx, const float* T, const float* Bx, const float* By, const float* Bz) {
  CTX_OR_RETURN(ctx);
  if (!c.staging) return fail(c, ASD_ESTATE, "asd_stage_fields_host: asd_set_staging has not been called");
  const size_t b = sizeof(float) * (size_t)c.N, pitch = align_up(b, 256) / sizeof(float);
  // the previous commit's pack kernels must have read the staging area before it is overwritten
  ASD_CUDA_TRY(c, cudaStreamWaitEvent(c.copy_stream, c.consumed_ev, 0));
  const float* src[4] = {T, Bx, By, Bz};
  for (int a = 0; a < 4; ++a) {
    if (!src[a]) continue;
    ASD_CUDA_TRY(c, cudaMemcpyAsync(c.staging + (size_t)a * pitch, src[a], b, cudaMemcpyHostToDevice, c.copy_stream));
    c.staged_mask |= 1u << a;
  }
  ASD_CUDA_TRY(c, cudaEventRecord(c.staged_ev, c.copy_stream));
  return ASD_OK;
}

asd_status asd_commit_fields(asd_ctx* ctx) {
  CTX_OR_RETURN(ctx);
  if (!c.staging) return fail(c, ASD_ESTATE, "asd_commit_fields: asd_set_staging has not been called");
  if (!c.staged_mask) return ASD_OK;
  const size_t pitch = align_up(sizeof(float) * (size_t)c.N, 256) / sizeof(float);
  ASD_CUDA_TRY(c, cudaStreamWaitEvent(c.stream, c.staged_ev, 0));
  const float* st = c.staging;
  const asd_status r = set_fields_impl(c, (c.staged_mask & 1u) ? st : nullptr, (c.staged_mask & 2u) ? st + pitch : nullptr,
                                       (c.staged_mask & 4u) ? st + 2 * pitch : nullptr,
                                       (c.staged_mask & 8u) ? st + 3 * pitch : nullptr, false);
  c.staged_mask = 0;
  ASD_CUDA_TRY(c, cudaEventRecord(c.consumed_ev, c.stream));
  return r;
}

asd_status asd_set_field_scale(asd_ctx* ctx, float s) {
  CTX_OR_RETURN(ctx);
  if (!std::isfinite(s)) return fail(c, ASD_EINVAL, "asd_set_field_scale: not finite");
  c.scale = s;
  return ASD_OK;
}

asd_status asd_step_heun(asd_ctx* ctx, int64_t n) {
  CTX_OR_RETURN(ctx);
  if (n < 0) return fail(c, ASD_EINVAL, "asd_step_heun: n < 0");
  return launch_heun(c, n);
}

asd_status asd_set_kernel(asd_ctx* ctx, int32_t variant) {
  CTX_OR_RETURN(ctx);
  if (variant != ASD_KERNEL_AUTO && variant != ASD_KERNEL_GENERAL && variant != ASD_KERNEL_FAST &&
      variant != ASD_KERNEL_TMA && variant != ASD_KERNEL_FUSED && variant != ASD_KERNEL_PERSISTENT)
    return fail(c, ASD_EINVAL, "asd_set_kernel: unknown variant");
  if (variant == ASD_KERNEL_PERSISTENT && !heun_persist_supported(c))
    return fail(c, ASD_EUNSUPPORTED, "asd_set_kernel: the persistent cluster needs built-in shells, ny % 4 == 0, grains that do not touch, no demagnetising field or meshes, and x-slabs that fit a CTA");
  if (variant == ASD_KERNEL_FUSED && (!heun_fused_supported(c) || (c.demag && c.demag_every < 1) || !fused_plan(c)))
    return fail(c, ASD_EUNSUPPORTED, "asd_set_kernel: the fused step needs what the film kernel needs, a strip plan that fits in shared memory, and -- with the demagnetising field on -- the held-field scheme (asd_set_demag_every >= 1)");
  if (variant == ASD_KERNEL_TMA && edge_field_on(c)) return fail(c, ASD_EUNSUPPORTED, "asd_set_kernel: the staged film kernel takes neither a multiscale window nor track-coupled ends");
  if (variant == ASD_KERNEL_TMA && (!heun_tma_supported(c) || !tma_plan(c)))
    return fail(c, ASD_EUNSUPPORTED, "asd_set_kernel: the staged film kernel needs what the film kernel needs and a strip plan that fits in shared memory");
  if (variant == ASD_KERNEL_FAST && !heun_fast_supported(c))
    return fail(c, ASD_EUNSUPPORTED, "asd_set_kernel: the film kernel needs open boundaries, ny % 4 == 0, built-in shells and grains that do not touch");
  c.kernel_variant = variant;
  graphs_invalidate(c);
  return ASD_OK;
}

asd_status asd_set_graph_mode(asd_ctx* ctx, int32_t mode) {
  CTX_OR_RETURN(ctx);
  if (mode != ASD_GRAPH_AUTO && mode != ASD_GRAPH_OFF && mode != ASD_GRAPH_ON)
    return fail(c, ASD_EINVAL, "asd_set_graph_mode: unknown mode");
  c.graph_mode = mode;
  return ASD_OK;
}

size_t asd_demag_workspace_bytes(asd_ctx* ctx) {
  if (!ctx) return 0;
  return demag_workspace_bytes(ctx->c);
}

asd_status asd_enable_demag(asd_ctx* ctx, const double spacing_m[3], void* d_workspace, size_t bytes) {
  CTX_OR_RETURN(ctx);
  if (!spacing_m || !(spacing_m[0] > 0.0) || !(spacing_m[1] > 0.0) || !(spacing_m[2] > 0.0))
    return fail(c, ASD_EINVAL, "asd_enable_demag: lattice constants must be > 0");
  if (!d_workspace || ((uintptr_t)d_workspace & 255u)) return fail(c, ASD_EINVAL, "asd_enable_demag: workspace NULL or not 256-byte aligned");
  if (c.d.ell_width > 0 || c.d.pbc[0] || c.d.pbc[1] || c.d.pbc[2])
    return fail(c, ASD_EUNSUPPORTED, "asd_enable_demag: open-boundary lattices with built-in shells only");
  c.demag_age = 0;
  return demag_enable(c, spacing_m, d_workspace, bytes);
}

asd_status asd_set_demag_every(asd_ctx* ctx, int32_t every) {
  CTX_OR_RETURN(ctx);
  if (every < 0) return fail(c, ASD_EINVAL, "asd_set_demag_every: every < 0");
  c.demag_every = every;
  c.demag_age = 0;
  return ASD_OK;
}

asd_status asd_demag_field(asd_ctx* ctx, float* cells, int64_t dims[3]) {
  CTX_OR_RETURN(ctx);
  if (!dims) return fail(c, ASD_EINVAL, "asd_demag_field: dims is NULL");
  if (!c.demag) return fail(c, ASD_ESTATE, "asd_demag_field: asd_enable_demag has not been called");
  return demag_field_host(c, cells, dims);
}

asd_status asd_demag_held_field(asd_ctx* ctx, float* cells, int64_t dims[3]) {
  CTX_OR_RETURN(ctx);
  if (!dims) return fail(c, ASD_EINVAL, "asd_demag_held_field: dims is NULL");
  if (!c.demag) return fail(c, ASD_ESTATE, "asd_demag_held_field: asd_enable_demag has not been called");
  return demag_field_host(c, cells, dims, true);
}

size_t asd_track_exchange_workspace_bytes(const asd_ctx* ctx) { return ctx ? track_exchange_workspace_bytes(ctx->c) : 0; }

asd_status asd_enable_track_exchange(asd_ctx* ctx, int32_t on, void* d_workspace, size_t bytes) {
  CTX_OR_RETURN(ctx);
  if (c.d.ell_width > 0 || c.d.pbc[0]) return fail(c, ASD_EUNSUPPORTED, "asd_enable_track_exchange: built-in shells, open in x");
  if (c.kernel_variant == ASD_KERNEL_TMA) return fail(c, ASD_EUNSUPPORTED, "asd_enable_track_exchange: not with ASD_KERNEL_TMA");
  if (on && (!d_workspace || ((uintptr_t)d_workspace & 255u)))
    return fail(c, ASD_EINVAL, "asd_enable_track_exchange: workspace NULL or not 256-byte aligned");
  graphs_invalidate(c);
  return track_exchange_enable(c, on, d_workspace, bytes);
}

size_t asd_track_stray_workspace_bytes(asd_ctx* ctx, int32_t range_cells) {
  if (!ctx) return 0;
  return demag_stray_workspace_bytes(ctx->c, range_cells);
}

asd_status asd_enable_track_stray(asd_ctx* ctx, int32_t on, int32_t range_cells, void* d_workspace, size_t bytes) {
  CTX_OR_RETURN(ctx);
  if (!c.demag) return fail(c, ASD_ESTATE, "asd_enable_track_stray: asd_enable_demag has not been called");
  if (on && (!d_workspace || ((uintptr_t)d_workspace & 255u)))
    return fail(c, ASD_EINVAL, "asd_enable_track_stray: workspace NULL or not 256-byte aligned");
  return demag_stray_enable(c, on, range_cells, d_workspace, bytes);
}

asd_status asd_track_stray_field(asd_ctx* ctx, float* cells) {
  CTX_OR_RETURN(ctx);
  if (!cells) return fail(c, ASD_EINVAL, "asd_track_stray_field: cells is NULL");
  if (!demag_stray_on(c)) return fail(c, ASD_ESTATE, "asd_track_stray_field: asd_enable_track_stray has not been called");
  return demag_stray_field_host(c, cells);
}

// the track's stray field belongs to one window origin and one track state
static asd_status then_refresh_stray(Ctx& c, asd_status st) {
  if (st == ASD_OK) st = demag_stray_refresh(c);
  if (st == ASD_OK) st = track_exchange_refresh(c);
  return st;
}

asd_status asd_shift_window(asd_ctx* ctx, int32_t p) {
  CTX_OR_RETURN(ctx);
  if (p < 1 || p > c.d.nx) return fail(c, ASD_EINVAL, "asd_shift_window: p must be in 1..nx");
  if (c.d.ell_width > 0) return fail(c, ASD_EUNSUPPORTED, "asd_shift_window: a general ELL table cannot follow the window");
  if (c.d.pbc[0]) return fail(c, ASD_EUNSUPPORTED, "asd_shift_window: window is periodic in x");
  if (c.x0 + p + c.d.nx > c.d.track_nx) return fail(c, ASD_ESTATE, "asd_shift_window: past the end of the track");
  graphs_invalidate(c);                        // window origin and buffer roles are frozen in recorded graphs
  demag_held_invalidate(c);                             // a held demagnetising field belongs to the old window position
  if (c.mm) {                                  // multiscale window: whole cells, through the meshes (M10)
    int64_t dl[3], dr[3];
    mm_dims(c, 0, dl); mm_dims(c, 1, dr);
    const int mx = c.d.macro[0];
    if (p % mx != 0 || p / mx > dl[0] || p / mx > dr[0])
      return fail(c, ASD_EINVAL, "asd_shift_window: a multiscale window moves by whole macrocells, at most the shorter mesh");
    if ((c.x0 + c.d.nx) / mx + dr[0] + p / mx > c.ncx) return fail(c, ASD_ESTATE, "asd_shift_window: leading mesh past the end of the track");
    return then_refresh_stray(c, launch_shift_mm(c, p));
  }
  return then_refresh_stray(c, launch_shift(c, p));
}

asd_status asd_magnetisation(asd_ctx* ctx, double m[3], double* n_magnetic) {
  CTX_OR_RETURN(ctx);
  if (!m) return fail(c, ASD_EINVAL, "asd_magnetisation: m is NULL");
  double o[4];
  const asd_status s = launch_magnetisation(c, o);
  if (s != ASD_OK) return s;
  const double inv = o[3] > 0.0 ? 1.0 / o[3] : 0.0;
  m[0] = o[0] * inv; m[1] = o[1] * inv; m[2] = o[2] * inv;
  if (n_magnetic) *n_magnetic = o[3];
  return ASD_OK;
}

asd_status asd_magnetisation_planes(asd_ctx* ctx, int32_t i0, int32_t n, double sum[3], double* n_magnetic) {
  CTX_OR_RETURN(ctx);
  if (!sum) return fail(c, ASD_EINVAL, "asd_magnetisation_planes: sum is NULL");
  if (i0 < 0 || n < 1 || (int64_t)i0 + n > c.d.nx) return fail(c, ASD_EINVAL, "asd_magnetisation_planes: planes outside the window");
  double o[4];
  const asd_status s = launch_magnetisation(c, o, i0, n);
  if (s != ASD_OK) return s;
  sum[0] = o[0]; sum[1] = o[1]; sum[2] = o[2];
  if (n_magnetic) *n_magnetic = o[3];
  return ASD_OK;
}

asd_status asd_planes_view(asd_ctx* ctx, int32_t comp, int32_t i0, int32_t n, float** d_ptr, size_t* count) {
  CTX_OR_RETURN(ctx);
  if (!d_ptr || !count) return fail(c, ASD_EINVAL, "asd_planes_view: NULL output pointer");
  if (comp < 0 || comp > 2 || i0 < 0 || n < 1 || (int64_t)i0 + n > c.d.nx)
    return fail(c, ASD_EINVAL, "asd_planes_view: component must be 0..2 and the planes inside the window");
  const size_t planep = (size_t)c.d.nz * (size_t)c.nyp;
  *d_ptr = c.arr(c.aS + comp) + c.lead + (size_t)i0 * planep;
  *count = (size_t)n * planep;
  demag_held_invalidate(c);                             // the caller is about to change spins behind the library's back
  mm_restart_cadence(c);
  return ASD_OK;
}

asd_status asd_grain_magnetisation(asd_ctx* ctx, double* m) {
  CTX_OR_RETURN(ctx);
  if (!m) return fail(c, ASD_EINVAL, "asd_grain_magnetisation: m is NULL");
  return launch_grain_magnetisation(c, m);
}

asd_status asd_track_dims(const asd_ctx* ctx, int64_t dims[3]) {
  if (!ctx || !dims) return ASD_EINVAL;
  dims[0] = ctx->c.ncx; dims[1] = ctx->c.ncy; dims[2] = ctx->c.ncz;
  return ASD_OK;
}

asd_status asd_track_set_init(asd_ctx* ctx, const float* mean_spin, float m0) {
  CTX_OR_RETURN(ctx);
  const size_t n = 3 * (size_t)c.ncell;
  float* im = nullptr;
  ASD_CUDA_TRY(c, cudaMallocHost(&im, sizeof(float) * n));
  for (int64_t q = 0; q < c.ncell; ++q)
    for (int a = 0; a < 3; ++a) im[3 * q + a] = mean_spin ? mean_spin[3 * q + a] : (a == 2 ? m0 : 0.0f);
  cudaError_t e = cudaMemcpyAsync(c.init_mean, im, sizeof(float) * n, cudaMemcpyHostToDevice, c.stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c.stream);
  cudaFreeHost(im);
  if (e != cudaSuccess) return fail_cuda(c, e, "asd_track_set_init copy");
  return then_refresh_stray(c, launch_cell_frames(c));
}

asd_status asd_track_get(asd_ctx* ctx, double* sum, int64_t* count) {
  CTX_OR_RETURN(ctx);
  if (sum) ASD_CUDA_TRY(c, cudaMemcpyAsync(sum, c.out_sum, sizeof(double) * 3 * (size_t)c.ncell, cudaMemcpyDeviceToHost, c.stream));
  if (count) ASD_CUDA_TRY(c, cudaMemcpyAsync(count, c.out_cnt, sizeof(long long) * (size_t)c.ncell, cudaMemcpyDeviceToHost, c.stream));
  ASD_CUDA_TRY(c, cudaStreamSynchronize(c.stream));
  return ASD_OK;
}

asd_status asd_track_end_pass(asd_ctx* ctx) {
  CTX_OR_RETURN(ctx);
  if (c.d.ell_width > 0) return fail(c, ASD_EUNSUPPORTED, "asd_track_end_pass: a general ELL table has no track");
  return then_refresh_stray(c, launch_track_end_pass(c));
}

asd_status asd_track_begin_pass(asd_ctx* ctx, int64_t x0_new) {
  CTX_OR_RETURN(ctx);
  if (c.d.ell_width > 0) return fail(c, ASD_EUNSUPPORTED, "asd_track_begin_pass: a general ELL table cannot follow the window");
  if (c.d.pbc[0]) return fail(c, ASD_EUNSUPPORTED, "asd_track_begin_pass: window is periodic in x");
  if (x0_new < 0 || x0_new + c.d.nx > c.d.track_nx) return fail(c, ASD_EINVAL, "asd_track_begin_pass: window must lie inside the track");
  if (c.mm) {
    int64_t dl[3], dr[3];
    mm_dims(c, 0, dl); mm_dims(c, 1, dr);
    const int mx = c.d.macro[0];
    if (x0_new % mx != 0 || x0_new / mx - dl[0] < 0 || (x0_new + c.d.nx) / mx + dr[0] > c.ncx)
      return fail(c, ASD_EINVAL, "asd_track_begin_pass: a multiscale window starts on a whole macrocell with both meshes inside the track");
  }
  graphs_invalidate(c);
  demag_held_invalidate(c);
  return then_refresh_stray(c, launch_track_begin_pass(c, x0_new));
}

asd_status asd_track_read_scan(asd_ctx* ctx, double y_r, double sigma_x, double sigma_y, double x_first, double x_step,
                               int64_t count, double* out) {
  CTX_OR_RETURN(ctx);
  if (!out || count < 1) return fail(c, ASD_EINVAL, "asd_track_read_scan: out is NULL or count < 1");
  if (!(sigma_x > 0.0) || !(sigma_y > 0.0) || !std::isfinite(sigma_x) || !std::isfinite(sigma_y) || !std::isfinite(y_r) ||
      !std::isfinite(x_first) || !std::isfinite(x_step))
    return fail(c, ASD_EINVAL, "asd_track_read_scan: footprint widths must be > 0 and positions finite");
  return launch_track_read_scan(c, y_r, sigma_x, sigma_y, x_first, x_step, count, out);
}

static const char* mm_check(const Ctx& c, const asd_mm_desc* d) {
  if (!d || !d->K0 || !d->Tc || !d->cell_grain) return "asd_mm: NULL description or array";
  if (d->mcx[0] < 1 || d->mcx[1] < 1 || d->every < 1) return "asd_mm: mcx[] and every must be >= 1";
  if (!(d->Ms0 > 0.0) || !std::isfinite(d->Ms0)) return "asd_mm: Ms0 must be > 0";
  for (int a = 0; a < 3; ++a) {
    if (!(d->A0[a] >= 0.0) || !std::isfinite(d->A0[a])) return "asd_mm: A0[] must be >= 0";
    if (!(d->spacing_m[a] > 0.0)) return "asd_mm: lattice constants must be > 0";
  }
  const int mx = c.d.macro[0];
  if (c.x0 % mx != 0 || c.d.nx % mx != 0) return "asd_mm: window origin and length must be whole macrocells";
  if (c.x0 / mx - d->mcx[0] < 0 || (c.x0 + c.d.nx) / mx + d->mcx[1] > c.ncx) return "asd_mm: meshes must lie inside the track";
  for (int g = 0; g < c.d.n_grains; ++g)
    if (!(d->Tc[g] > 0.0) || !std::isfinite(d->K0[g])) return "asd_mm: Tc[] must be > 0 and K0[] finite";
  for (int64_t t = 0; t < c.ncx * c.ncy; ++t)
    if (d->cell_grain[t] < -1 || d->cell_grain[t] >= c.d.n_grains) return "asd_mm: cell grain id out of range";
  return nullptr;
}

size_t asd_mm_workspace_bytes(const asd_ctx* ctx, const asd_mm_desc* desc) {
  if (!ctx || !desc || desc->mcx[0] < 1 || desc->mcx[1] < 1) return 0;
  return mm_workspace_bytes(ctx->c, desc->mcx);
}

asd_status asd_mm_enable(asd_ctx* ctx, const asd_mm_desc* desc, void* d_workspace, size_t bytes) {
  CTX_OR_RETURN(ctx);
  if (c.d.ell_width > 0 || c.d.pbc[0] || c.d.pbc[1] || c.d.pbc[2])
    return fail(c, ASD_EUNSUPPORTED, "asd_mm_enable: open-boundary lattices with built-in shells only");
  if (c.kernel_variant == ASD_KERNEL_TMA) return fail(c, ASD_EUNSUPPORTED, "asd_mm_enable: not with ASD_KERNEL_TMA");
  if (const char* why = mm_check(c, desc)) return fail(c, ASD_EINVAL, why);
  if (!d_workspace || ((uintptr_t)d_workspace & 255u)) return fail(c, ASD_EINVAL, "asd_mm_enable: workspace NULL or not 256-byte aligned");
  graphs_invalidate(c);
  return mm_enable(c, *desc, d_workspace, bytes);
}

asd_status asd_mm_dims(const asd_ctx* ctx, int32_t side, int64_t dims[3]) {
  if (!ctx || !dims || (side != 0 && side != 1)) return ASD_EINVAL;
  if (!ctx->c.mm) return ASD_ESTATE;
  mm_dims(ctx->c, side, dims);
  return ASD_OK;
}

#define MM_OR_RETURN(name)                                                                         \
  if (side != 0 && side != 1) return fail(c, ASD_EINVAL, name ": side must be 0 or 1");            \
  if (!c.mm) return fail(c, ASD_ESTATE, name ": asd_mm_enable has not been called");

asd_status asd_mm_set_fields_host(asd_ctx* ctx, int32_t side, const float* T, const float* Bx, const float* By, const float* Bz) {
  CTX_OR_RETURN(ctx);
  MM_OR_RETURN("asd_mm_set_fields_host");
  return mm_set_fields_host(c, side, T, Bx, By, Bz);
}

asd_status asd_mm_set_m_host(asd_ctx* ctx, int32_t side, const float* m) {
  CTX_OR_RETURN(ctx);
  MM_OR_RETURN("asd_mm_set_m_host");
  if (!m) return fail(c, ASD_EINVAL, "asd_mm_set_m_host: m is NULL");
  return mm_set_m_host(c, side, m);
}

asd_status asd_mm_get_m_host(asd_ctx* ctx, int32_t side, float* m) {
  CTX_OR_RETURN(ctx);
  MM_OR_RETURN("asd_mm_get_m_host");
  if (!m) return fail(c, ASD_EINVAL, "asd_mm_get_m_host: m is NULL");
  return mm_get_m_host(c, side, m);
}

asd_status asd_get_counters(const asd_ctx* ctx, int64_t* step, int64_t* shift, int64_t* x0, int64_t* pass) {
  if (!ctx) return ASD_EINVAL;
  if (step) *step = ctx->c.step;
  if (shift) *shift = ctx->c.shift;
  if (x0) *x0 = ctx->c.x0;
  if (pass) *pass = ctx->c.pass;
  return ASD_OK;
}

asd_status asd_set_counters(asd_ctx* ctx, int64_t step, int64_t shift, int64_t pass) {
  CTX_OR_RETURN(ctx);
  if (step < 0 || shift < 0 || pass < 0) return fail(c, ASD_EINVAL, "asd_set_counters: negative counter");
  c.step = step; c.shift = shift; c.pass = pass;
  return ASD_OK;
}

int64_t asd_launch_count(const asd_ctx* ctx) { return ctx ? ctx->c.launches : 0; }

const char* asd_last_error(const asd_ctx* ctx) {
  if (ctx && ctx->c.err[0]) return ctx->c.err;
  return g_static_err;
}

const char* asd_version(void) { return "asd-b200 0.1 (sm_100a)"; }

}  // extern "C"
