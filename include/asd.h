/* ============================================================================
 * asd.h -- C ABI of libasd: the atomistic spin-dynamics (ASD) window of the multiscale HAMR
 * model of arXiv 2502.02236 (Gija et al.), as hand-written CUDA kernels for NVIDIA B200 (sm_100a).
 *
 * Citations: P:<n> = PAPER.md line n (with section / equation); S:<x> = SURVEY.md section 8 item x;
 * D:<x> = DESIGN.md reading x.
 *
 * What the library computes
 *   * stochastic Landau-Lifshitz-Gilbert equation on every atomic spin, Eq. (1) (sec. II)
 *   * effective field B = mu_0 H in Tesla: exchange Eq. (2) + uniaxial anisotropy Eq. (3)
 *      + external (write) field + thermal field, sigma = sqrt(2 lambda k_B T /
 *     (gamma mu_s dt)) (P:38 with mu_0 absorbed)
 *   * stochastic Heun integration (BASELINE.json north_star; D:Q1), noise from Philox4x32-10 keyed by
 *     (seed; step, global site) generated in registers (D:R1-R3)
 *   * moving-window shift: outgoing slab -> track macrocells by Eq. (6), incoming
 *     slab <- cone sampling about the track magnetisation (D:S3)
 *   * window / per-grain magnetisation (Eq. (6) with V = window or grain)
 *
 * Conventions
 *   Site order   window-local l = (i*nz + k)*ny + j; x (i) along the track and slowest, z (k) film normal,
 *                y (j) across the track and fastest.  All per-site arrays are [N], N = nx*ny*nz, fp32.
 *   Global id    g = l + x0*ny*nz -- the Philox counter, so noise follows the atom, not the memory slot.
 *   Units        Tesla, Joule, Kelvin, seconds; mu_s in J/T; gamma in rad s^-1 T^-1.
 *   Pointers     "DEVICE" = CUDA device memory on the context's device; "HOST" = ordinary host memory
 *                (pinned memory makes the *_host calls asynchronous; pageable memory makes them
 *                synchronise).  The caller owns every buffer it passes.  The library copies what it
 *                needs into the caller-provided workspace and never frees or keeps a caller pointer
 *                except `d_workspace` (which must outlive the context).
 *   Streams      every call enqueues on the `cuda_stream` given at create time and returns without
 *                synchronising, except asd_magnetisation, asd_grain_magnetisation, asd_track_get,
 *                asd_get_spins_host (they synchronise that stream).
 *   Errors       every call returns asd_status.  Arguments are validated on the host -> ASD_EINVAL.
 *                A CUDA failure is sticky: the context returns ASD_ECUDA until destroyed.
 *                asd_last_error gives a static or context-owned message.  No exceptions, no abort().
 *   Threads      a context is not thread-safe; distinct contexts are independent.
 *   No fallback  there is no CPU path: without a CUDA device asd_create_lattice returns ASD_ECUDA.
 * ========================================================================== */
#ifndef ASD_H_
#define ASD_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define ASD_API __attribute__((visibility("default")))
#else
#define ASD_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct asd_ctx asd_ctx; /* opaque; created by asd_create_lattice, freed by asd_destroy */

typedef enum {
  ASD_OK = 0,
  ASD_EINVAL = 1,       /* bad argument (null, size, range)                                   */
  ASD_ENOMEM = 2,       /* workspace too small                                                */
  ASD_ECUDA = 3,        /* CUDA runtime / launch failure (sticky)                             */
  ASD_ESTATE = 4,       /* call not valid in the current state (e.g. shift past the track end)*/
  ASD_EUNSUPPORTED = 5  /* valid request the library does not implement                       */
} asd_status;

enum { ASD_SC = 0, ASD_L10_FE = 1 };

/* Kernel variant for asd_step_heun.  AUTO picks the fastest supported.
 * FUSED: one kernel per Heun step (predictor results stay in shared memory / registers); FAST, TMA, GENERAL: one
 * kernel per stage; PERSISTENT: all n steps of an asd_step_heun(n) call in one launch of one thread-block cluster that
 * keeps the lattice in (distributed) shared memory -- 16 CTAs where the device schedules that cluster size, else 8; x-slabs
 * of at most 1024 four-site groups that fit a CTA's shared memory, built-in shells, grains that do not touch; what AUTO
 * runs where it measured faster than graph replay (slabs of up to 1024-3072 sites per CTA, by lattice). */
enum { ASD_KERNEL_AUTO = 0, ASD_KERNEL_GENERAL = 1, ASD_KERNEL_FAST = 2, ASD_KERNEL_TMA = 3, ASD_KERNEL_FUSED = 4,
       ASD_KERNEL_PERSISTENT = 5 };

/* CUDA-graph replay of asd_step_heun batches (launch-bound lattices).  AUTO: on for windows of <= 2^18 sites. */
enum { ASD_GRAPH_AUTO = 0, ASD_GRAPH_OFF = 1, ASD_GRAPH_ON = 2 };

/* Lattice description (S:8(b)).  Plain data; HOST pointers are read during asd_create_lattice only. */
typedef struct {
  int32_t lattice;      /* ASD_SC: simple cubic, 6 nearest neighbours, J[0]
                           ASD_L10_FE: Fe sublattice of L1_0 FePt in its own simple-tetragonal axes,
                           4 in-plane nn J[0] at (+-1,0,0),(0,+-1,0); 2 out-of-plane J[1] at (0,0,+-1);
                           4 in-plane nnn J[2] at (+-1,+-1,0)  ("4 nearest + 6 next nearest") */
  int32_t nx, ny, nz;   /* window size in sites                                                  */
  int32_t pbc[3];       /* periodic flags (x,y,z); a periodic dimension needs n >= 3 (D:Q17);
                           pbc[0] requires track_nx == nx and forbids asd_shift_window            */
  double mu_s;          /* atomic moment, J/T                                                    */
  double lambda;        /* Gilbert damping, >= 0                                                 */
  double gamma;         /* gyromagnetic ratio, rad s^-1 T^-1; <= 0 selects 1.76085963023e11       */
  double dt;            /* time step, s, > 0                                                     */
  double J[3];          /* exchange energies per shell, Joule (see `lattice`)                    */
  int64_t track_nx;     /* length of the grain map in planes, >= x0 + nx                         */
  int64_t x0;           /* global plane index of window plane 0                                  */
  const int32_t *grain_map; /* HOST [track_nx*ny], grain id of column (gx, j) at gx*ny + j; -1 = vacant
                               (non-magnetic) column.  NULL = one grain (id 0) everywhere.
                               Exchange bonds join only magnetic sites of the SAME grain.   */
  int32_t n_grains;     /* >= 1, <= 65535                                                        */
  const float *grain_ku;   /* HOST [n_grains] uniaxial anisotropy energy per atom K_1, Joule (Eq. 3); NULL = 0 */
  const float *grain_axis; /* HOST [n_grains*3] unit easy axes e_A (|e| = 1 within 1e-4); NULL = z */
  int32_t macro[3];     /* track macrocell edge in sites (mx,my,mz), each >= 1 (D:S1)            */
  const int32_t *ell_idx;  /* optional general neighbour table, HOST [N*ell_width] site-major, entry =
                              window-local neighbour site or -1; replaces the built-in shells      */
  const float *ell_J;      /* HOST [N*ell_width] exchange energy of that pair, Joule              */
  int32_t ell_width;    /* 0 = built-in shells; else 1..16                                       */
  uint64_t seed;        /* Philox key                                                            */
} asd_lattice_desc;

/* Bytes of DEVICE workspace asd_create_lattice needs for this description (0 if desc is invalid).
 * Callable without a GPU. */
ASD_API size_t asd_workspace_bytes(const asd_lattice_desc *desc);

/* Creates a context.  d_workspace: DEVICE, >= asd_workspace_bytes(desc) bytes, 256-byte aligned, owned by
 * the caller and kept until asd_destroy.  cuda_stream: a cudaStream_t (NULL = default stream).
 * Initial state: all spins +z on magnetic sites (0 on vacant), T = 0, B = 0, field scale 1, counters 0,
 * track initial state +z with m0 = 1.  ASD_EINVAL / ASD_ENOMEM / ASD_ECUDA. */
ASD_API asd_status asd_create_lattice(const asd_lattice_desc *desc, void *d_workspace, size_t bytes,
                              void *cuda_stream, asd_ctx **out);
ASD_API asd_status asd_destroy(asd_ctx *ctx);

/* Spins, SoA fp32 [N] each.  set: values on vacant sites are ignored (stored as 0); values are NOT
 * renormalised.  get: vacant sites read 0. */
ASD_API asd_status asd_set_spins(asd_ctx *ctx, const float *sx, const float *sy, const float *sz);      /* DEVICE */
ASD_API asd_status asd_get_spins(asd_ctx *ctx, float *sx, float *sy, float *sz);                        /* DEVICE */
ASD_API asd_status asd_set_spins_host(asd_ctx *ctx, const float *sx, const float *sy, const float *sz); /* HOST */
ASD_API asd_status asd_get_spins_host(asd_ctx *ctx, float *sx, float *sy, float *sz);       /* HOST; synchronises */

/* Per-site temperature T [K] and applied field B [Tesla] in window-local order (the profiles
 * are centred in the window and do not move with a shift).  NULL = keep the previous array.
 * T < 0 is the caller's error (sigma becomes NaN); it is not scanned. */
ASD_API asd_status asd_set_fields(asd_ctx *ctx, const float *T, const float *Bx, const float *By,
                          const float *Bz);                                                     /* DEVICE */
ASD_API asd_status asd_set_fields_host(asd_ctx *ctx, const float *T, const float *Bx, const float *By,
                               const float *Bz);                                                /* HOST   */
/* B_app = s * B : write-field polarity / ramp. */
ASD_API asd_status asd_set_field_scale(asd_ctx *ctx, float s);

/* Double-buffered upload of host fields, for callers that change T / B every batch (the laser and the head move):
 * the host-to-device copy of the NEXT batch's fields overlaps the Heun steps of the current one.
 *   asd_set_staging        once: a caller-owned DEVICE buffer of asd_staging_bytes(ctx) bytes, 256-byte aligned.
 *   asd_stage_fields_host  starts the copy of the given HOST arrays (pinned for a truly asynchronous copy; NULL = leave
 *                          that field as it is) into the staging buffer on an internal stream and returns at once; the
 *                          arrays must stay valid and unchanged until the next asd_commit_fields has been called and
 *                          the stream has passed it.  It first waits (on the device) for the previous commit.
 *   asd_commit_fields      makes the staged fields the current ones for every step enqueued after it (the context's
 *                          stream waits for the copy, then repacks as asd_set_fields does).  Nothing staged: no-op.
 * ASD_ESTATE before asd_set_staging. */
ASD_API size_t asd_staging_bytes(const asd_ctx *ctx);
ASD_API asd_status asd_set_staging(asd_ctx *ctx, void *d_staging, size_t bytes);
ASD_API asd_status asd_stage_fields_host(asd_ctx *ctx, const float *T, const float *Bx, const float *By, const float *Bz);
ASD_API asd_status asd_commit_fields(asd_ctx *ctx);

/* n stochastic Heun steps (S:O4): per step one predictor and one corrector kernel, each fused
 * field + update + renormalise with in-register Philox noise (same xi in both stages); step counter += n. */
ASD_API asd_status asd_step_heun(asd_ctx *ctx, int64_t n);
/* Selects the kernel variant (ASD_KERNEL_*); ASD_EUNSUPPORTED if the lattice cannot use it. */
ASD_API asd_status asd_set_kernel(asd_ctx *ctx, int32_t variant);
/* Selects whether asd_step_heun(n >= 2) replays recorded CUDA graphs (ASD_GRAPH_*).  Results do not depend on it. */
ASD_API asd_status asd_set_graph_mode(asd_ctx *ctx, int32_t mode);

/* ---- Demagnetising field of the window (Eq. (6)-(7)) ----------------------------------
 * Once enabled, every Heun stage adds to the effective field of a site the field of its track macrocell,
 *   B_c = -mu_0 sum_c' N(r_c' - r_c) M_c',  M_c = (mu_s / V) sum_{j in c} S_j   (V = macro[0..2] * spacing, full cell),
 * N = demagnetising tensor of two equal cuboids (Newell et al., the paper's ref. [28]), summed over the macrocells that
 * overlap the window (open boundaries).  Open-boundary lattices with the built-in shells; ASD_KERNEL_TMA and CUDA graphs
 * are not used while it is on; ASD_KERNEL_FUSED (and AUTO's choice of it) needs the held-field scheme of
 * asd_set_demag_every (every >= 1).  The caller owns the workspace (DEVICE, 256-byte aligned) for the life of the context.
 * The convolution is the library's own (direct sum over the film's macrocell layers, DFT across the film, shared-memory
 * FFT along the track; no FFT library): ASD_EUNSUPPORTED if 3 * (layers of macrocells) fields of the padded track length
 * do not fit in one CTA's shared memory (about 300 macrocell layers x cells along x / 256).
 * asd_demag_workspace_bytes is pure host arithmetic.  asd_demag_field computes the field of the current
 * spins per macrocell into HOST cells[dims[0]*dims[1]*dims[2]*3] (x-cell slowest, component fastest; Tesla) and
 * synchronises; cells == NULL returns dims only.  ASD_ESTATE if demag is not enabled. */
ASD_API size_t asd_demag_workspace_bytes(asd_ctx *ctx);
ASD_API asd_status asd_enable_demag(asd_ctx *ctx, const double spacing_m[3], void *d_workspace, size_t bytes);
ASD_API asd_status asd_demag_field(asd_ctx *ctx, float *cells, int64_t dims[3]);
/* every == 0 (default): the field is recomputed from the configuration of EVERY Heun stage (exact Heun on the full
 * field).  every = P >= 1: it is recomputed from S at the predictor of every P-th Heun step (counted from the last
 * enable / this call / window shift / asd_set_spins) and held for both stages in between (reading D3). */
ASD_API asd_status asd_set_demag_every(asd_ctx *ctx, int32_t every);
/* The cell field as the last Heun stage used it (nothing is recomputed): in the held-field scheme, the field of the
 * spins at the last refresh.  Same HOST layout, dims and errors as asd_demag_field; synchronises.  With the one-kernel
 * step (ASD_KERNEL_FUSED / AUTO) the macrocell sums of Eq. (6) behind a refresh are accumulated by the corrector of the
 * step before it (64-bit fixed point, order-independent), not by a pass of their own over the spins. */
ASD_API asd_status asd_demag_held_field(asd_ctx *ctx, float *cells, int64_t dims[3]);

/* Window ends exchange coupled to the frozen track ("the ends of the simulation window are exchange coupled to the
 * track"; reading E1), for a purely atomistic window (the meshes of asd_mm_enable take the ends over).  The
 * neighbour spins beyond the first / last plane in Eq. (2) -- x-1 of plane 0, x+1 of plane nx-1, for L1_0 their two
 * in-plane diagonals as well -- are the DIRECTION of the frozen track in the macrocell that holds the neighbour position
 * (what the window has written there, else what lies ahead; as for a micromagnetic neighbour), subject to the
 * same-grain rule.  Off by default (the ends are then open boundaries).  Recomputed whenever the window origin or the
 * track store changes.  Caller-owned DEVICE workspace (256-byte aligned) for the life of the context.  Not with general
 * ELL tables, pbc[0], ASD_KERNEL_TMA, ASD_KERNEL_PERSISTENT, CUDA-graph replay. */
ASD_API size_t asd_track_exchange_workspace_bytes(const asd_ctx *ctx);
ASD_API asd_status asd_enable_track_exchange(asd_ctx *ctx, int32_t on, void *d_workspace, size_t bytes);

/* Stray field of the frozen track on the window ("the stray field generated by [the frozen track] is fully
 * computed when the simulation window is shifted, and included in the simulation window at each iteration"; P:76;
 * DESIGN.md sec. 12, reading D4).  Needs asd_enable_demag (it shares the macrocell geometry and rides on the cell field
 * the Heun kernels already add).  Sources: of every track macrocell, the sites that are NOT inside the window --
 *   mom_c' = out_sum_c' (what has left the window: the frozen spins themselves)
 *          + init_mean_c' * (magnetic sites of the cell the window has never held),     M_c' = (mu_s / V) mom_c',
 *   B_c = -mu_0 sum_c' N(r_c' - r_c) M_c'   over the track cells within range_cells of the target cell along x
 *                                           (range_cells <= 0: the whole track),
 * with the cuboid tensor of asd_enable_demag; a cell the window edge cuts is a source with its outside sites.  The field
 * is recomputed (two small kernels, direct sum) at enable time and whenever the window origin or the track store
 * changes: asd_shift_window, asd_track_set_init, asd_track_end_pass, asd_track_begin_pass.  Caller-owned DEVICE
 * workspace (256-byte aligned) for the life of the context; on == 0 switches it off.  asd_track_stray_field copies the
 * field per window macrocell to HOST cells[dims[0]*dims[1]*dims[2]*3] (layout of asd_demag_field) and synchronises.
 * ASD_ESTATE without asd_enable_demag. */
ASD_API size_t asd_track_stray_workspace_bytes(asd_ctx *ctx, int32_t range_cells);
ASD_API asd_status asd_enable_track_stray(asd_ctx *ctx, int32_t on, int32_t range_cells, void *d_workspace, size_t bytes);
ASD_API asd_status asd_track_stray_field(asd_ctx *ctx, float *cells);

/* Window moves +x by p planes, 1 <= p <= nx (S:O5): outgoing planes -> macrocell sums and counts (Eq. 6);
 * spins move by p planes; incoming planes seeded by cone sampling (D:S3); x0 += p; shift counter += 1.
 * ASD_ESTATE if x0 + p + nx > track_nx; ASD_EUNSUPPORTED with a general ELL table or pbc[0]. */
ASD_API asd_status asd_shift_window(asd_ctx *ctx, int32_t p_planes);

/* m = sum over magnetic sites of S / N_mag (Eq. 6 with V = window), fp64; synchronises. */
ASD_API asd_status asd_magnetisation(asd_ctx *ctx, double m[3], double *n_magnetic);
/* Per-grain mean spin, HOST [n_grains*3] (0 for grains without sites in the window); synchronises. */
ASD_API asd_status asd_grain_magnetisation(asd_ctx *ctx, double *m);

/* Track store: macrocells (cx,cy,cz) = (floor(gx/mx), floor(j/my), floor(k/mz)), cell index
 * c = (cx*ncy + cy)*ncz + cz over the whole track. */
ASD_API asd_status asd_track_dims(const asd_ctx *ctx, int64_t dims[3]);
/* What lies ahead of the window: mean spin per cell, HOST [ncell*3] (|v| <= 1 is the reduced
 * magnetisation M/M_S^0); NULL = (0,0,m0) everywhere. */
ASD_API asd_status asd_track_set_init(asd_ctx *ctx, const float *mean_spin, float m0);
/* What the window has written: sum of spins and site count per cell (Eq. 6 with mu_S/V factored out).
 * HOST sum [ncell*3] (fp64), count [ncell]; either may be NULL; synchronises. */
ASD_API asd_status asd_track_get(asd_ctx *ctx, double *sum, int64_t *count);

/* ---- Passes over the track: writing parallel tracks one after the other (sec. III / Fig. 4: "The written
 * bit pattern was then used as the starting state for a second pass through the track shifting algorithm"; DESIGN.md
 * sec. 13, readings T1-T3) -----------------------------------------------------------------------------------------------
 * asd_track_end_pass    the nx planes still inside the window are transferred to the track by Eq. (6) exactly
 *                       as outgoing planes are; then every macrocell the pass has written (count > 0) becomes what lies
 *                       ahead of the next pass: init mean spin = sum / count (cells never written keep theirs).  The
 *                       written store stays readable (asd_track_get, asd_track_read_scan).  Asynchronous.  The window's
 *                       spins now belong to the track as well: start the next pass (or load new spins) before stepping
 *                       on with the demagnetising / stray field, which would otherwise count them twice.
 * asd_track_begin_pass  the written store is cleared, pass counter += 1, the window returns to global plane x0_new
 *                       (0 <= x0_new <= track_nx - nx) and ALL its planes are generated from the track by the cone
 *                       sampling of P:68 (D:S3) with Philox counter n := pass; step and shift counters run on.  T and B
 *                       are not touched.  Asynchronous.  ASD_EUNSUPPORTED with a general ELL table or pbc[0].
 * asd_track_read_scan   read-back figure of merit standing in for the TMR read head of P:114: the mean S_z per magnetic
 *                       site of the WRITTEN store under a Gaussian reader footprint,
 *                         R(x_r) = sum_c w_c sum_z[c] / sum_c w_c count[c],
 *                         w_c = exp(-(x_c - x_r)^2 / (2 sigma_x^2) - (y_c - y_r)^2 / (2 sigma_y^2)),
 *                       (x_c, y_c) = ((cx + 1/2) mx, (cy + 1/2) my) the nominal centre of macrocell c in site units (x in
 *                       global planes), all layers cz summed; x_r = x_first + n x_step, n = 0 .. count-1; 0 where the
 *                       footprint holds no written site.  out: HOST [count] fp64; deterministic; synchronises. */
ASD_API asd_status asd_track_end_pass(asd_ctx *ctx);
ASD_API asd_status asd_track_begin_pass(asd_ctx *ctx, int64_t x0_new);
ASD_API asd_status asd_track_read_scan(asd_ctx *ctx, double y_r, double sigma_x, double sigma_y, double x_first,
                                       double x_step, int64_t count, double *out);

/* ---- Multiscale window: micromagnetic LLG meshes either side of the atomistic mesh (Fig. 1, P:29-33, P:38, P:54-62,
 * P:118, readings M1-M10) --------------------------------------------------------------------------
 * The window becomes [trailing mesh | atomistic mesh | leading mesh]; the mesh cells are the track macrocells, so the
 * window origin x0 and nx must be whole cells (multiples of macro[0]) and the meshes must lie inside the track.
 *   state      one unit direction m per cell (0 = empty cell), fp32
 *   field      B = (2 A_0 m_e / M_S^0) lap(m) + (2 K_0 m_e^2 / M_S^0)(m.e)e + s B_app     (Eq. (4), (5) with A = A_0 m_e^2,
 *              K = K_0 m_e^3, M_S = M_S^0 m_e; 6-neighbour stencil; none between different grains);
 *              m_e(T) = largest root of m = B(3 T_C m / T + mu_s |s B_app| / k_B T), B(x) = coth x - 1/x
 *   dynamics   Eq. (1) without the stochastic field, damping lambda (1 - T / 3 T_C) (held at its T_C value above
 *              T_C), classical RK4: one step of every * dt per `every` Heun steps
 *   coupling   across each mesh boundary, both ways: the atomistic sites of the first / last plane take the
 *              mesh direction in place of their missing neighbour spins in Eq. (2); the mesh cells take the direction
 *              of the average atomistic spin of the adjacent stencil cell in the Laplacian; the far mesh ends take the
 *              frozen track.  Boundary data is exchanged when the meshes step and held in between.
 *   shift      asd_shift_window then moves by whole cells (p a multiple of macro[0], at most the shorter mesh):
 *              trailing mesh -> track store (as m_e m per magnetic site), outgoing atoms -> trailing mesh by Eq. (6),
 *              leading mesh -> incoming atoms by the cone sampling of P:68 about m with magnitude m_e, track ahead ->
 *              leading mesh; ASD_EINVAL otherwise.
 * HOST pointers of the description are read during asd_mm_enable only.  The caller owns the workspace (DEVICE, 256-byte
 * aligned) for the life of the context.  Not available with general ELL tables, periodic boundaries, ASD_KERNEL_TMA,
 * CUDA-graph replay (ASD_EUNSUPPORTED).
 *   passes     asd_track_end_pass also transfers every cell of both meshes to the track store (as m_e m on the cell's
 *              magnetic sites); asd_track_begin_pass(x0_new) needs x0_new on a whole macrocell with both meshes inside
 *              the track, and restarts the meshes along the track they then lie over. */
typedef struct {
  int32_t mcx[2];            /* cells along x of the trailing / leading mesh, each >= 1                          */
  int32_t every;             /* Heun steps per RK4 step, >= 1                                                    */
  double Ms0;                /* M_S^0, A/m                                                                       */
  double A0[3];              /* A_0 along x, y, z, J/m (one value three times = the paper's scalar A)            */
  const double *K0;          /* HOST [n_grains] K_0, J/m^3 (easy axes = grain_axis of the lattice)               */
  const double *Tc;          /* HOST [n_grains] T_C, K                                                           */
  const int32_t *cell_grain; /* HOST [ncx*ncy] grain id of track cell column (cx, cy) at cx*ncy + cy; -1 = empty */
  double spacing_m[3];       /* lattice constants, metres (cell edge = macro * spacing)                          */
} asd_mm_desc;
ASD_API size_t asd_mm_workspace_bytes(const asd_ctx *ctx, const asd_mm_desc *desc);
/* Initial mesh state: the direction of the track the meshes lie over; T = 0, B = 0. */
ASD_API asd_status asd_mm_enable(asd_ctx *ctx, const asd_mm_desc *desc, void *d_workspace, size_t bytes);
/* dims = (mcx[side], ncy, ncz); cell (a, b, c) of a mesh is element (a*ncy + b)*ncz + c of the arrays below. */
ASD_API asd_status asd_mm_dims(const asd_ctx *ctx, int32_t side, int64_t dims[3]);
/* Per-cell temperature [K] and applied field [Tesla] of one mesh, HOST [cells]; window-fixed profiles like the
 * atomistic ones; NULL = keep.  Synchronises. */
ASD_API asd_status asd_mm_set_fields_host(asd_ctx *ctx, int32_t side, const float *T, const float *Bx, const float *By,
                                          const float *Bz);
/* Cell directions of one mesh, HOST [cells*3] (component fastest).  set: empty cells stay 0.  Both synchronise. */
ASD_API asd_status asd_mm_set_m_host(asd_ctx *ctx, int32_t side, const float *m);
ASD_API asd_status asd_mm_get_m_host(asd_ctx *ctx, int32_t side, float *m);

/* ---- Slab decomposition across devices ("implemented for ... multiple GPUs"; DESIGN.md
 * sec. 9) --------------------------------------------------------------------------------------------------------------
 * A window cut along x into slabs is just one ordinary context per slab whose window holds the slab's own planes plus
 * H >= 2 ghost planes towards each neighbour: one Heun step spoils two more ghost planes from the outside in (the
 * predictor of a plane needs its x neighbours, the corrector the predictor of its x neighbours), so H ghost planes last
 * H / 2 steps, and the own planes stay exact -- the noise is keyed by GLOBAL site, so a slab computes for a ghost atom
 * what its owner computes.  Between steps the owners' planes are copied over the ghosts; these two calls are what that
 * copy needs, and nothing else in the library knows about slabs (paper_2502_02236_b200/slab.py drives it: device-to-
 * device copies between contexts of one process, or NCCL send/recv between ranks).
 *   asd_planes_view            DEVICE pointer to the storage of planes i0 .. i0+n-1 of component comp (0, 1, 2) of the
 *                              CURRENT spins: *count = n * nz * row_stride floats, contiguous, rows of ny sites at the
 *                              library's padded row stride (the pad floats are zero and must stay zero; two contexts
 *                              with equal ny and nz have equal strides, so planes are copied verbatim).  The pointer is
 *                              valid until the next asd_step_heun / asd_shift_window / asd_set_spins on this context
 *                              (the spins change buffers): ask again after each.  Writing through it is the caller's
 *                              responsibility: vacant sites must receive zeros (a peer's copy of the same planes does).
 *   asd_magnetisation_planes   sum of S over the magnetic sites of planes i0 .. i0+n-1 and their number (fp64, same
 *                              deterministic reduction as asd_magnetisation); synchronises. */
ASD_API asd_status asd_planes_view(asd_ctx *ctx, int32_t comp, int32_t i0, int32_t n, float **d_ptr, size_t *count);
ASD_API asd_status asd_magnetisation_planes(asd_ctx *ctx, int32_t i0, int32_t n, double sum[3], double *n_magnetic);

/* ---- A reduction that allocates nothing (csrc/asd_noalloc.cu) --------------------------------------------------------
 * For callers that cannot call cudaMalloc or hand over a workspace: code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid allocation.  Needs no context.  The deterministic two-stage reduction of asd_magnetisation
 * (Eq. (6)) over three DEVICE arrays of `count` floats each -- e.g. what asd_planes_view hands out; pad floats
 * and vacant sites hold exact zeros -- written to DEVICE d_out4[4] = (sum S_x, sum S_y, sum S_z, number of elements that
 * hold a spin: |S|^2 > 1/4), fp64.  Enqueued on cuda_stream (a cudaStream_t, NULL = default stream) of the CURRENT
 * device; does not synchronise; the caller owns inputs and output.
 * Its partial sums live in a static 64 KB array in device memory that every GPU loading the library holds until the
 * process exits; hence count <= ASD_NOALLOC_MAX_COUNT (ASD_EINVAL beyond, also for NULL pointers or count == 0; message
 * from asd_last_error(NULL)).  Every call on a device shares that array: calls that overlap on the GPU (different
 * streams without an event between them) race; calls in one stream do not.  ASD_ECUDA without a device. */
#define ASD_NOALLOC_MAX_COUNT 8388608
ASD_API asd_status asd_spin_sum_noalloc(const float *d_sx, const float *d_sy, const float *d_sz, size_t count,
                                        double *d_out4, void *cuda_stream);

/* Counters for bit-exact checkpoint / resume (Philox is counter based: there is no RNG state). */
ASD_API asd_status asd_get_counters(const asd_ctx *ctx, int64_t *step, int64_t *shift, int64_t *x0, int64_t *pass);
ASD_API asd_status asd_set_counters(asd_ctx *ctx, int64_t step, int64_t shift, int64_t pass);

/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
ASD_API int64_t asd_launch_count(const asd_ctx *ctx);

/* Message of the last failure on this context (or a generic one for ctx == NULL); never NULL. */
ASD_API const char *asd_last_error(const asd_ctx *ctx);
/* Library version string, e.g. "asd-b200 0.1 (sm_100a)". */
ASD_API const char *asd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ASD_H_ */
