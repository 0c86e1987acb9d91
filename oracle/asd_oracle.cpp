// ============================================================================
// oracle/asd_oracle.cpp -- plain fp64 CPU oracle for the atomistic spin-dynamics
// (ASD) window of arXiv 2502.02236 (Gija et al., multiscale HAMR model).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
// header, table or constant generator with the CUDA library under
// paper_2502_02236_b200/csrc/ and neither includes the other.
//
// What it computes, and where the definition comes from (P:<n> = /root/reference/PAPER.md
// line n; S:<x> = SURVEY.md section 8(c) item x; D:<x> = DESIGN.md reading x):
//   * stochastic LLG, Eq. (1), P:35          -> llg_rhs()          (LL form, S:O4)
//   * thermal field sigma, P:38               -> sigma_T()          (Tesla units, S:O3)
//   * exchange field Eq. (2), P:46-48         -> field_at()
//   * uniaxial anisotropy Eq. (3), P:50-52    -> field_at()
//   * stochastic Heun step                    -> orc_step_heun()    (S:O4, BASELINE north_star)
//   * atomistic->macrocell transfer Eq. (6), P:64-66 -> orc_shift_window() outgoing part
//   * macrocell->atomistic cone thermalisation, P:68 -> seed_site()  (S:S3 reading)
//   * Philox4x32-10 (Salmon et al., SC'11, public definition) -> philox4x32_10()
//   * multiscale window: micromagnetic LLG meshes either side of the atomistic mesh, Eq. (4)-(5), temperature scalings
//     m_e(T), A = A0 m_e^2, K = K0 m_e^3, alpha = lambda (1 - T/3T_C), RK4, two-way exchange coupling
//     across the mesh boundaries, transfers on a shift (Fig. 1) -> the "Multiscale window" section (S:8(f) item 3)
//   * stray field of the frozen track on the window -> stray_cells()  (reading D4)
//   * passes over the track (two parallel tracks) -> orc_track_end_pass(), orc_track_begin_pass();
//     Gaussian-footprint read-back standing in for the TMR head -> orc_track_read_scan()  (S:8(f) item 4)
//
// Everything is written in the paper's order and notation, one site at a time, with
// explicit coordinate loops; no blocking, fusion or reordering.  OpenMP is used only
// over sites inside one Jacobi stage (each site reads the OLD configuration), which does
// not change any result.
//
// Units: B = mu_0 H in Tesla, energies in Joule, mu_s in J/T, gamma in rad s^-1 T^-1.
//
// Pins (tests/test_oracle_*.py; table in DESIGN.md sec. 3): Philox vs ATen host engine; single-spin damped
// precession closed form; Langevin function; monotone energy; brute-force energy
// gradient; |S|=1; spin-wave dispersion (fixes exchange normalisation and the L1_0
// shell geometry); simple-cubic T_C = 1.44 J/k_B;
// shift index exactness; seeded-slab magnetisation magnitude (P:68 purpose clause);
// cuboid demagnetising tensor vs direct quadrature and sum rules (P12); track stray field vs the
// whole-track field (D4); ELL branch, magnetisation divisors, held-field composition (round 2);
// track passes and read-back scan (T1-T3); m_e(T), macrospin with alpha(T), RK4 order, mesh spin
// waves, both directions of the mesh coupling, whole-cell shift (P13-P19).
// "parity unpinned": the OUTCOME of a recording run (which grains end up reversed) and
// the paper's TMR read-head signal (its solver is not part of the method; orc_track_read_scan
// is a stated stand-in and is pinned as such).
// ============================================================================
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kBoltzmann = 1.380649e-23;  // J/K (SI exact)

// ---------------------------------------------------------------------------
// Philox4x32-10.  Public definition: Salmon, Moraes, Dror, Shaw, SC'11.
// One round: (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
// M0 = 0xD2511F53, M1 = 0xCD9E8D57; key bumped by (0x9E3779B9, 0xBB67AE85) between rounds.
// ---------------------------------------------------------------------------
void philox4x32_10(const uint32_t key_in[2], const uint32_t ctr_in[4], uint32_t out[4]) {
  uint32_t k0 = key_in[0], k1 = key_in[1];
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) {
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// S:R1 keying.  key = (seed lo, seed hi); counter = (n lo, n hi, g lo, g hi | stream<<28).
// n = step index before the step (thermal noise) or the pass number (shift seeding);
// g = GLOBAL site id (gx*nz + k)*ny + j, so noise follows the atom, not the memory slot.
void philox_block(uint64_t seed, uint64_t n, uint64_t g, uint32_t stream, uint32_t out[4]) {
  const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {(uint32_t)(n & 0xFFFFFFFFull), (uint32_t)(n >> 32),
                           (uint32_t)(g & 0xFFFFFFFFull), (uint32_t)(g >> 32) | (stream << 28)};
  philox4x32_10(key, ctr, out);
}

// S:R2.  u = ((r >> 9) + 1/2) * 2^-23 in (0,1); exactly representable in fp32 and fp64.
inline double uniform_from_u32(uint32_t r) { return ((double)(r >> 9) + 0.5) * (1.0 / 8388608.0); }

// S:R3.  Box-Muller: xi_x = rho0 cos(2 pi u1), xi_y = rho0 sin(2 pi u1), rho0 = sqrt(-2 ln u0);
// xi_z = rho2 cos(2 pi u3), rho2 = sqrt(-2 ln u2).  The fourth normal is discarded.
void normals3(uint64_t seed, uint64_t step, uint64_t g, double xi[3]) {
  uint32_t r[4];
  philox_block(seed, step, g, 0u, r);
  const double u0 = uniform_from_u32(r[0]), u1 = uniform_from_u32(r[1]);
  const double u2 = uniform_from_u32(r[2]), u3 = uniform_from_u32(r[3]);
  const double rho0 = std::sqrt(-2.0 * std::log(u0));
  const double rho2 = std::sqrt(-2.0 * std::log(u2));
  xi[0] = rho0 * std::cos(2.0 * kPi * u1);
  xi[1] = rho0 * std::sin(2.0 * kPi * u1);
  xi[2] = rho2 * std::cos(2.0 * kPi * u3);
}

// theta_max = root in [0, pi] of sin(theta)/theta = m  (S:S3: the distribution P:68 states --
// polar angle uniform on [0, theta_max], free azimuth -- has <cos theta> = sin(theta_max)/theta_max,
// so this root is what "reproduces the correct magnetization magnitude M").
double theta_max_of_m(double m) {
  if (m >= 1.0) return 0.0;
  if (m <= 0.0) return kPi;
  double lo = 0.0, hi = kPi;  // sin(x)/x decreases monotonically from 1 to 0 on [0, pi]
  for (int it = 0; it < 200; ++it) {
    const double mid = 0.5 * (lo + hi);
    const double v = (mid == 0.0) ? 1.0 : std::sin(mid) / mid;
    if (v > m) lo = mid; else hi = mid;
  }
  return 0.5 * (lo + hi);
}

struct Oracle {
  int lattice = 0;               // 0 = simple cubic, 1 = L1_0 Fe sublattice (simple tetragonal axes)
  int nx = 0, ny = 0, nz = 0;    // x along track, z film normal
  int pbc[3] = {0, 0, 0};
  double mu_s = 0, lambda = 0, gamma = 0, dt = 0;
  double J[3] = {0, 0, 0};
  int64_t track_nx = 0, x0 = 0;
  std::vector<int32_t> grain_map;  // [track_nx * ny], -1 = vacant column
  int n_grains = 0;
  std::vector<double> ku;          // [n_grains]  J per atom
  std::vector<double> axis;        // [n_grains*3]
  int macro[3] = {1, 1, 1};
  int ell_width = 0;               // > 0: general ELL override
  std::vector<int32_t> ell_idx;    // [N * ell_width] site-major, -1 = none
  std::vector<double> ell_J;       // [N * ell_width] Joule
  uint64_t seed = 0;
  int64_t step = 0, shift = 0, pass = 0;
  double scale = 1.0;              // B_app = scale * B
  int64_t N = 0;
  std::vector<double> sx, sy, sz;  // spins (0 on vacant sites)
  std::vector<double> T, Bx, By, Bz;
  // track store (macrocells over the whole track)
  int64_t ncx = 0, ncy = 0, ncz = 0;
  std::vector<double> out_sum;     // [ncell*3]  sum of m_j (Eq. 6 with mu_S/V factored out)
  std::vector<int64_t> out_cnt;    // [ncell]
  std::vector<double> init_mean;   // [ncell*3]  what lies ahead of the window
  int threads = 0;
  // demagnetising field (Eq. (6)-(7)); off unless orc_enable_demag was called
  bool demag = false;
  double cell_m[3] = {0, 0, 0};    // macrocell edge lengths, metres
  int dcx = 0, dcy = 0, dcz = 0;   // macrocells that can overlap the window (x: worst alignment)
  std::vector<double> demag_N;     // [(2dcx-1)(2dcy-1)(2dcz-1)][6]: Nxx Nyy Nzz Nxy Nxz Nyz at cell offsets
  int demag_every = 0;             // 0: recomputed in every stage; P >= 1: from S at every P-th step, held in between (D3)
  int64_t demag_age = 0;           // steps since the held field was invalidated (enable, set_every, shift, set_spins)
  std::vector<double> demag_hold;  // the held per-macrocell field
  // stray field of the frozen track on the window's macrocells (reading D4); off unless enabled
  bool track_exch = false;         // window ends exchange coupled to the frozen track (reading E1); off unless enabled
  bool stray = false;
  int stray_range = 0;             // source cells taken up to this many cells from a target cell along x; 0 = the whole track
  bool stray_dirty = true;         // window origin or track state changed since stray_B was computed
  std::vector<double> stray_B;     // [dcx*dcy*dcz*3] Tesla
  // multiscale window (S:8(f) item 3): micromagnetic LLG meshes either side of the atomistic
  // mesh; off unless orc_mm_enable was called.  Mesh cells ARE track macrocells; side 0 = trailing (lower x), 1 = leading.
  bool mm = false;
  struct MicroMesh {
    int mcx = 0;                          // cells along x
    std::vector<double> m;                // [mcx*ncy*ncz*3] unit magnetisation direction; 0 for an empty cell
    std::vector<double> T, Bx, By, Bz;    // per cell, window-fixed profiles
    std::vector<double> me, alpha;        // m_e(T) and alpha(T) per cell
  } mesh[2];
  double mm_Ms0 = 0, mm_A0[3] = {0, 0, 0};  // M_S^0 [A/m]; A_0 [J/m] along x, y, z (one value three times = the paper's scalar A)
  std::vector<double> mm_K0, mm_Tc;       // per grain: K_0 [J/m^3], T_C [K]
  std::vector<int32_t> mm_grain;          // [ncx*ncy] grain id of a track cell column (cx, cy), -1 = empty
  double mm_cell[3] = {0, 0, 0};          // cell edge lengths, metres
  int mm_every = 1;                       // Heun steps per RK4 step: dt_mm = mm_every * dt
  int64_t mm_age = 0;                     // Heun steps since the last (re)start of the exchange cadence
  std::vector<double> mm_ghost[2];        // [ncy*ncz*3] direction of the mesh cells that touch the atomistic mesh (held)
  std::vector<double> mm_avg[2];          // [ncy*ncz*3] direction of the average atomistic spin in the stencil cell (held)

  int64_t site(int i, int k, int j) const { return ((int64_t)i * nz + k) * ny + j; }
  int32_t grain_of(int i, int j) const { return grain_map[(size_t)((x0 + i) * ny + j)]; }
  int64_t cell_of(int64_t gx, int j, int k) const {
    return ((gx / macro[0]) * ncy + (j / macro[1])) * ncz + (k / macro[2]);
  }
};

// sigma_i = sqrt(2 lambda k_B T_i / (gamma mu_s dt))  [Tesla]; P:38 with mu_0 absorbed (B = mu_0 H).
inline double sigma_T(const Oracle& o, double T) {
  return std::sqrt(2.0 * o.lambda * kBoltzmann * T / (o.gamma * o.mu_s * o.dt));
}

// Neighbour shells (S:O3).  SC: 6 nn, J[0].  L1_0 Fe sublattice in its own simple-tetragonal
// axes: 4 in-plane nn J[0], 2 out-of-plane J[1], 4 in-plane nnn J[2] ("4 nearest + 6 next nearest",
// z = 10; geometry fixed by A_L10 = 3J/2a, see the spin-wave pin).
struct Offset { int dx, dy, dz, shell; };
const Offset kOffsetsSC[6] = {{1,0,0,0},{-1,0,0,0},{0,1,0,0},{0,-1,0,0},{0,0,1,0},{0,0,-1,0}};
const Offset kOffsetsL10[10] = {{1,0,0,0},{-1,0,0,0},{0,1,0,0},{0,-1,0,0},
                                {0,0,1,1},{0,0,-1,1},
                                {1,1,0,2},{1,-1,0,2},{-1,1,0,2},{-1,-1,0,2}};

// Wrap or reject a coordinate.  Returns false when the neighbour does not exist (open boundary).
inline bool wrap(int& c, int n, int periodic) {
  if (c >= 0 && c < n) return true;
  if (!periodic) return false;
  c = (c % n + n) % n;
  return true;
}

bool track_direction(const Oracle& o, int64_t cx, int b, int c, double n[3]);   // defined with the multiscale window

// Exchange sum  sum_j J_ij X_j  (Joule), Eq. (2) numerator, for site (i,k,j) in configuration X.
// A bond is kept only if the neighbour exists, both ends are magnetic and in the same grain
// (exchange-decoupled grains).
void exchange_sum(const Oracle& o, const double* X0, const double* X1, const double* X2,
                  int i, int k, int j, double e[3]) {
  e[0] = e[1] = e[2] = 0.0;
  const int64_t l = o.site(i, k, j);
  if (o.ell_width > 0) {
    for (int s = 0; s < o.ell_width; ++s) {
      const int32_t n = o.ell_idx[(size_t)(l * o.ell_width + s)];
      if (n < 0) continue;
      const double Jij = o.ell_J[(size_t)(l * o.ell_width + s)];
      e[0] += Jij * X0[n]; e[1] += Jij * X1[n]; e[2] += Jij * X2[n];
    }
    return;
  }
  const int32_t g = o.grain_of(i, j);
  const Offset* offs = (o.lattice == 0) ? kOffsetsSC : kOffsetsL10;
  const int noff = (o.lattice == 0) ? 6 : 10;
  for (int s = 0; s < noff; ++s) {
    int ii = i + offs[s].dx, jj = j + offs[s].dy, kk = k + offs[s].dz;
    if (!o.mm && o.track_exch && !o.pbc[0] && (ii == -1 || ii == o.nx)) {
      // Reading E1 ("the ends of the simulation window are exchange coupled to the track"): the neighbour spin beyond
      // the window's first / last plane is the DIRECTION of the frozen track in the macrocell that holds the neighbour
      // position (what the window has written there, else what lies ahead) -- as for a micromagnetic neighbour.
      const int64_t gxn = o.x0 + ii;
      if (gxn < 0 || gxn >= o.track_nx || jj < 0 || jj >= o.ny || kk < 0 || kk >= o.nz) continue;
      const int32_t gn = o.grain_map[(size_t)(gxn * o.ny + jj)];
      if (gn < 0 || gn != g) continue;                        // exchange-decoupled grains
      double nd[3];
      if (!track_direction(o, gxn / o.macro[0], jj / o.macro[1], kk / o.macro[2], nd)) continue;
      const double Jij = o.J[offs[s].shell];
      e[0] += Jij * nd[0]; e[1] += Jij * nd[1]; e[2] += Jij * nd[2];
      continue;
    }
    if (o.mm && (ii == -1 || ii == o.nx)) {
      // Across the mesh boundary: "For the contribution from the micromagnetic region the respective
      // magnetization direction is used directly" -- the neighbour spin of Eq. (2) is the direction m of the
      // micromagnetic cell that holds the neighbour position (as captured at the last exchange, reading M9).
      if (jj < 0 || jj >= o.ny || kk < 0 || kk >= o.nz) continue;
      const int32_t gn = o.grain_map[(size_t)((o.x0 + ii) * o.ny + jj)];
      if (gn < 0 || gn != g) continue;                        // exchange-decoupled grains
      const double* mg = &o.mm_ghost[ii < 0 ? 0 : 1][3 * ((size_t)(jj / o.macro[1]) * o.ncz + kk / o.macro[2])];
      const double Jij = o.J[offs[s].shell];
      e[0] += Jij * mg[0]; e[1] += Jij * mg[1]; e[2] += Jij * mg[2];
      continue;
    }
    if (!wrap(ii, o.nx, o.pbc[0])) continue;
    if (!wrap(jj, o.ny, o.pbc[1])) continue;
    if (!wrap(kk, o.nz, o.pbc[2])) continue;
    const int32_t gn = o.grain_of(ii, jj);
    if (gn < 0 || gn != g) continue;
    const int64_t n = o.site(ii, kk, jj);
    const double Jij = o.J[offs[s].shell];
    e[0] += Jij * X0[n]; e[1] += Jij * X1[n]; e[2] += Jij * X2[n];
  }
}

// ---- Demagnetising tensor of two equal cuboids (Newell, Williams and Dunlop, J. Geophys. Res. 98, 9551 (1993);
// the paper's ref. [28]): N_ab(R) such that the cell-averaged field of a uniformly magnetised source cell at
// offset R is H = -N M.  Written out as the 27-point second difference of the auxiliary functions f and g. ----
double newell_f(double x, double y, double z) {
  x = std::fabs(x); y = std::fabs(y); z = std::fabs(z);           // f is even in every argument
  const double x2 = x * x, y2 = y * y, z2 = z * z, R = std::sqrt(x2 + y2 + z2);
  if (R == 0.0) return 0.0;
  double v = (2.0 * x2 - y2 - z2) * R / 6.0;
  if (y > 0.0 && (x2 + z2) > 0.0) v += 0.5 * y * (z2 - x2) * std::asinh(y / std::sqrt(x2 + z2));
  if (z > 0.0 && (x2 + y2) > 0.0) v += 0.5 * z * (y2 - x2) * std::asinh(z / std::sqrt(x2 + y2));
  if (x > 0.0 && y > 0.0 && z > 0.0) v -= x * y * z * std::atan(y * z / (x * R));
  return v;
}
double newell_g(double x, double y, double z) {
  const double sgn = ((x < 0.0) != (y < 0.0)) ? -1.0 : 1.0;       // g is odd in x and in y, even in z
  x = std::fabs(x); y = std::fabs(y); z = std::fabs(z);
  const double x2 = x * x, y2 = y * y, z2 = z * z, R = std::sqrt(x2 + y2 + z2);
  if (R == 0.0) return 0.0;
  double v = -x * y * R / 3.0;
  if (z > 0.0 && (x2 + y2) > 0.0) v += x * y * z * std::asinh(z / std::sqrt(x2 + y2));
  if (x > 0.0 && (y2 + z2) > 0.0) v += y / 6.0 * (3.0 * z2 - y2) * std::asinh(x / std::sqrt(y2 + z2));
  if (y > 0.0 && (x2 + z2) > 0.0) v += x / 6.0 * (3.0 * z2 - x2) * std::asinh(y / std::sqrt(x2 + z2));
  if (z > 0.0) {
    if (x > 0.0 && y > 0.0) v -= z * z2 / 6.0 * std::atan(x * y / (z * R));
    if (y > 0.0 && x > 0.0) v -= 0.5 * z * y2 * std::atan(x * z / (y * R));
    if (x > 0.0 && y > 0.0) v -= 0.5 * z * x2 * std::atan(y * z / (x * R));
  }
  return sgn * v;
}
// sum_{u,v,w in {-1,0,1}} w_u w_v w_w F(X + u dx, Y + v dy, Z + w dz), w = (1, -2, 1)
template <class F>
double second_difference(F fn, double X, double Y, double Z, double dx, double dy, double dz) {
  static const double w[3] = {1.0, -2.0, 1.0};
  double acc = 0.0;
  for (int u = -1; u <= 1; ++u)
    for (int v = -1; v <= 1; ++v)
      for (int t = -1; t <= 1; ++t) acc += w[u + 1] * w[v + 1] * w[t + 1] * fn(X + u * dx, Y + v * dy, Z + t * dz);
  return acc;
}
// out = (Nxx, Nyy, Nzz, Nxy, Nxz, Nyz) for cell size d and offset R.  Beyond kDemagNear cell diagonals the second
// difference loses its digits to cancellation; there the cuboids are point dipoles to 1e-3 of an already tiny term:
// N_ab = V/(4 pi R^3) (delta_ab - 3 R_a R_b / R^2)   (reading D2).
constexpr double kDemagNear = 12.0;
void newell_tensor(const double d[3], const double Rv[3], double out[6]) {
  const double pi = 3.14159265358979323846;
  const double X = Rv[0], Y = Rv[1], Z = Rv[2], V = d[0] * d[1] * d[2];
  const double R2 = X * X + Y * Y + Z * Z, diag2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
  if (R2 > kDemagNear * kDemagNear * diag2) {
    const double R = std::sqrt(R2), c = V / (4.0 * pi * R2 * R);
    out[0] = c * (1.0 - 3.0 * X * X / R2); out[1] = c * (1.0 - 3.0 * Y * Y / R2); out[2] = c * (1.0 - 3.0 * Z * Z / R2);
    out[3] = -3.0 * c * X * Y / R2; out[4] = -3.0 * c * X * Z / R2; out[5] = -3.0 * c * Y * Z / R2;
    return;
  }
  const double k = -1.0 / (4.0 * pi * V);
  out[0] = k * second_difference(newell_f, X, Y, Z, d[0], d[1], d[2]);
  out[1] = k * second_difference(newell_f, Y, X, Z, d[1], d[0], d[2]);
  out[2] = k * second_difference(newell_f, Z, Y, X, d[2], d[1], d[0]);
  out[3] = k * second_difference(newell_g, X, Y, Z, d[0], d[1], d[2]);
  out[4] = k * second_difference(newell_g, X, Z, Y, d[0], d[2], d[1]);
  out[5] = k * second_difference(newell_g, Y, Z, X, d[1], d[2], d[0]);
}

// Demagnetising field of configuration X, Tesla, one 3-vector per window macrocell (S:8(f) item 1):
//   M_c = (mu_s / V) sum_{j in c} X_j                       Eq. (6), V = full macrocell volume
//   B_c = -mu_0 sum_c' N(r_c' - r_c) M_c'                    Eq. (7), open boundaries, the window's own cells only
// Cells are the track macrocells (global alignment): window cell (a,b,c) is track cell (x0/mx + a, b, c).
void demag_cells(const Oracle& o, const double* X0, const double* X1, const double* X2, std::vector<double>& Bd) {
  const double mu0 = 4.0e-7 * 3.14159265358979323846;
  const int mx = o.macro[0], my = o.macro[1], mz = o.macro[2];
  const int64_t c0 = o.x0 / mx;
  const int ncx = (int)((o.x0 + o.nx - 1) / mx - c0) + 1, ncy = o.dcy, ncz = o.dcz;
  const double V = o.cell_m[0] * o.cell_m[1] * o.cell_m[2];
  std::vector<double> M((size_t)ncx * ncy * ncz * 3, 0.0);
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        const int64_t l = o.site(i, k, j);
        const size_t c = ((size_t)((o.x0 + i) / mx - c0) * ncy + j / my) * ncz + k / mz;
        M[3 * c] += X0[l]; M[3 * c + 1] += X1[l]; M[3 * c + 2] += X2[l];
      }
  for (double& v : M) v *= o.mu_s / V;
  Bd.assign((size_t)o.dcx * ncy * ncz * 3, 0.0);
  const int sy = 2 * o.dcy - 1, sz = 2 * o.dcz - 1;
  for (int a = 0; a < ncx; ++a)
    for (int b = 0; b < ncy; ++b)
      for (int c = 0; c < ncz; ++c) {
        double H[3] = {0, 0, 0};
        for (int a2 = 0; a2 < ncx; ++a2)
          for (int b2 = 0; b2 < ncy; ++b2)
            for (int c2 = 0; c2 < ncz; ++c2) {
              const size_t t = (((size_t)(a2 - a + o.dcx - 1) * sy + (b2 - b + o.dcy - 1)) * sz + (c2 - c + o.dcz - 1)) * 6;
              const double* N = &o.demag_N[t];
              const double* m = &M[3 * (((size_t)a2 * ncy + b2) * ncz + c2)];
              H[0] -= N[0] * m[0] + N[3] * m[1] + N[4] * m[2];
              H[1] -= N[3] * m[0] + N[1] * m[1] + N[5] * m[2];
              H[2] -= N[4] * m[0] + N[5] * m[1] + N[2] * m[2];
            }
        const size_t q = 3 * (((size_t)a * ncy + b) * ncz + c);
        Bd[q] = mu0 * H[0]; Bd[q + 1] = mu0 * H[1]; Bd[q + 2] = mu0 * H[2];
      }
}
inline const double* demag_of_site(const Oracle& o, const std::vector<double>& Bd, int i, int k, int j) {
  const int64_t c0 = o.x0 / o.macro[0];
  const size_t c = ((size_t)((o.x0 + i) / o.macro[0] - c0) * o.dcy + j / o.macro[1]) * o.dcz + k / o.macro[2];
  return &Bd[3 * c];
}

// Stray field of the frozen track on the window's macrocells (reading D4; "the stray field generated by [the
// frozen track] is fully computed when the simulation window is shifted, and included in the simulation window at each
// iteration").  Sources: every track macrocell's sites that are NOT inside the window -- what has left it (out_sum,
// the actual frozen moments) and what the window has never held (init mean spin times the number of such magnetic sites):
//   mom_c' = out_sum_c' + init_mean_c' (n_behind_c' - out_cnt_c' + n_ahead_c'),   M_c' = (mu_s / V) mom_c'
//   B_c = -mu_0 sum_c' N(r_c' - r_c) M_c'      (Eq. (7) with the same cuboid tensor; a cell the window edge cuts is a
//                                               source with its outside sites and a demag cell with its inside sites)
void stray_cells(const Oracle& o, std::vector<double>& Bs) {
  const double mu0 = 4.0e-7 * 3.14159265358979323846;
  const int mx = o.macro[0], my = o.macro[1], mz = o.macro[2];
  const int64_t c0 = o.x0 / mx;
  const int ncxw = (int)((o.x0 + o.nx - 1) / mx - c0) + 1;
  const double V = o.cell_m[0] * o.cell_m[1] * o.cell_m[2];
  Bs.assign((size_t)o.dcx * o.dcy * o.dcz * 3, 0.0);
  for (int64_t cx = 0; cx < o.ncx; ++cx)
    for (int b2 = 0; b2 < o.ncy; ++b2)
      for (int c2 = 0; c2 < o.ncz; ++c2) {
        const size_t t = (size_t)((cx * o.ncy + b2) * o.ncz + c2);
        int64_t n_out = 0;                                   // magnetic sites of the cell outside the window
        const int kext = std::min((c2 + 1) * mz, o.nz) - c2 * mz;
        for (int64_t gx = cx * mx; gx < std::min<int64_t>((cx + 1) * mx, o.track_nx); ++gx) {
          if (gx >= o.x0 && gx < o.x0 + o.nx) continue;
          for (int j = b2 * my; j < std::min((b2 + 1) * my, o.ny); ++j)
            if (o.grain_map[(size_t)(gx * o.ny + j)] >= 0) n_out += kext;
        }
        const double fresh = (double)(n_out - o.out_cnt[t]);  // sites the window has never held
        double M[3];
        for (int u = 0; u < 3; ++u) M[u] = o.mu_s / V * (o.out_sum[3 * t + u] + o.init_mean[3 * t + u] * fresh);
        if (M[0] == 0.0 && M[1] == 0.0 && M[2] == 0.0) continue;
        for (int a = 0; a < ncxw; ++a) {
          if (o.stray_range > 0 && std::llabs(cx - (c0 + a)) > o.stray_range) continue;
          for (int b = 0; b < o.dcy; ++b)
            for (int c = 0; c < o.dcz; ++c) {
              const double R[3] = {(double)(cx - (c0 + a)) * o.cell_m[0], (double)(b2 - b) * o.cell_m[1], (double)(c2 - c) * o.cell_m[2]};
              double N[6];
              newell_tensor(o.cell_m, R, N);
              double* B = &Bs[3 * (((size_t)a * o.dcy + b) * o.dcz + c)];
              B[0] -= mu0 * (N[0] * M[0] + N[3] * M[1] + N[4] * M[2]);
              B[1] -= mu0 * (N[3] * M[0] + N[1] * M[1] + N[5] * M[2]);
              B[2] -= mu0 * (N[4] * M[0] + N[5] * M[1] + N[2] * M[2]);
            }
        }
      }
}
// cell field every site sees in a stage: the window's demagnetising field (Bd, already computed) + the track's stray field
void add_stray(Oracle& o, std::vector<double>& Bd) {
  if (!o.stray) return;
  if (o.stray_dirty) { stray_cells(o, o.stray_B); o.stray_dirty = false; }
  for (size_t t = 0; t < Bd.size(); ++t) Bd[t] += o.stray_B[t];
}

// Effective field in Tesla at a magnetic site (S:O3):
// B_i(X) = (1/mu_s) sum_j J_ij X_j + (2 k_u,g/mu_s)(X_i.e_g) e_g + s*B_app,i + sigma_i xi_i.
void field_at(const Oracle& o, const double* X0, const double* X1, const double* X2,
              int i, int k, int j, const double* xi /* may be null */, double B[3],
              const double* Bd = nullptr /* demagnetising field of the site's macrocell, or null */) {
  const int64_t l = o.site(i, k, j);
  const int32_t g = o.grain_of(i, j);
  double e[3];
  exchange_sum(o, X0, X1, X2, i, k, j, e);
  B[0] = e[0] / o.mu_s; B[1] = e[1] / o.mu_s; B[2] = e[2] / o.mu_s;        // Eq. (2)
  const double ex = o.axis[3 * g], ey = o.axis[3 * g + 1], ez = o.axis[3 * g + 2];
  const double d = X0[l] * ex + X1[l] * ey + X2[l] * ez;
  const double ca = 2.0 * o.ku[g] / o.mu_s * d;                             // Eq. (3)
  B[0] += ca * ex; B[1] += ca * ey; B[2] += ca * ez;
  B[0] += o.scale * o.Bx[l]; B[1] += o.scale * o.By[l]; B[2] += o.scale * o.Bz[l];
  if (Bd) { B[0] += Bd[0]; B[1] += Bd[1]; B[2] += Bd[2]; }                   // Eq. (7)
  if (xi) {
    const double sg = sigma_T(o, o.T[l]);
    B[0] += sg * xi[0]; B[1] += sg * xi[1]; B[2] += sg * xi[2];
  }
}

// f(S,B) = -gamma/(1+lambda^2) [ S x B + lambda S x (S x B) ]  -- Eq. (1) solved for dm/dt
// (cross Eq. (1) with m and use m.dm/dt = 0; S:O4).
inline void llg_rhs(const Oracle& o, const double S[3], const double B[3], double f[3]) {
  const double a0 = S[1] * B[2] - S[2] * B[1];
  const double a1 = S[2] * B[0] - S[0] * B[2];
  const double a2 = S[0] * B[1] - S[1] * B[0];
  const double b0 = S[1] * a2 - S[2] * a1;
  const double b1 = S[2] * a0 - S[0] * a2;
  const double b2 = S[0] * a1 - S[1] * a0;
  const double c = -o.gamma / (1.0 + o.lambda * o.lambda);
  f[0] = c * (a0 + o.lambda * b0);
  f[1] = c * (a1 + o.lambda * b1);
  f[2] = c * (a2 + o.lambda * b2);
}

// Threads for the per-stage site loops: the caller's choice, else all cores for large lattices and one
// for tiny ones (forking a team costs more than a few hundred sites of work).  Never changes a result.
inline int thread_count(const Oracle& o) {
#ifdef _OPENMP
  if (o.threads > 0) return o.threads;
  return o.N < 4096 ? 1 : omp_get_max_threads();
#else
  return 1;
#endif
}

// One stochastic Heun step, Jacobi order (S:O4):
// 1 draw xi_i; 2 k1 = f(S, B(S)); 3 S~ = (S + dt k1)/|.|; 4 k2 = f(S~, B(S~)) with the SAME xi_i;
// 5 S <- (S + dt/2 (k1+k2))/|.|; 6 n <- n+1.  Vacant sites are skipped and stay 0.
void mm_before_heun_step(Oracle& o);
void heun_step(Oracle& o) {
  const int64_t N = o.N;
  mm_before_heun_step(o);
  std::vector<double> xi(3 * (size_t)N, 0.0), k1(3 * (size_t)N, 0.0);
  std::vector<double> tx((size_t)N, 0.0), ty((size_t)N, 0.0), tz((size_t)N, 0.0);
  const int nx = o.nx, ny = o.ny, nz = o.nz;
  const int nt = thread_count(o);
  std::vector<double> Bd;                        // demagnetising field of the stage's configuration, per macrocell
  const bool held = o.demag && o.demag_every >= 1;
  if (held) {
    if (o.demag_age % o.demag_every == 0) demag_cells(o, o.sx.data(), o.sy.data(), o.sz.data(), o.demag_hold);
    Bd = o.demag_hold;
    o.demag_age += 1;
    add_stray(o, Bd);
  } else if (o.demag) {
    demag_cells(o, o.sx.data(), o.sy.data(), o.sz.data(), Bd);
    add_stray(o, Bd);
  }
#pragma omp parallel for collapse(2) schedule(static) num_threads(nt)
  for (int i = 0; i < nx; ++i)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j) {
        if (o.grain_of(i, j) < 0) continue;
        const int64_t l = o.site(i, k, j);
        const uint64_t g = (uint64_t)(((o.x0 + i) * nz + k) * ny + j);
        normals3(o.seed, (uint64_t)o.step, g, &xi[3 * l]);
        double B[3], f[3];
        field_at(o, o.sx.data(), o.sy.data(), o.sz.data(), i, k, j, &xi[3 * l], B,
                 o.demag ? demag_of_site(o, Bd, i, k, j) : nullptr);
        const double S[3] = {o.sx[l], o.sy[l], o.sz[l]};
        llg_rhs(o, S, B, f);
        k1[3 * l] = f[0]; k1[3 * l + 1] = f[1]; k1[3 * l + 2] = f[2];
        const double p0 = S[0] + o.dt * f[0], p1 = S[1] + o.dt * f[1], p2 = S[2] + o.dt * f[2];
        const double nrm = std::sqrt(p0 * p0 + p1 * p1 + p2 * p2);
        tx[l] = p0 / nrm; ty[l] = p1 / nrm; tz[l] = p2 / nrm;
      }
  std::vector<double> n0((size_t)N, 0.0), n1((size_t)N, 0.0), n2((size_t)N, 0.0);
  if (o.demag && !held) { demag_cells(o, tx.data(), ty.data(), tz.data(), Bd); add_stray(o, Bd); }   // B(S~): demagnetising field of S~ (+ the track's)
#pragma omp parallel for collapse(2) schedule(static) num_threads(nt)
  for (int i = 0; i < nx; ++i)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j) {
        if (o.grain_of(i, j) < 0) continue;
        const int64_t l = o.site(i, k, j);
        double B[3], f[3];
        field_at(o, tx.data(), ty.data(), tz.data(), i, k, j, &xi[3 * l], B,
                 o.demag ? demag_of_site(o, Bd, i, k, j) : nullptr);
        const double St[3] = {tx[l], ty[l], tz[l]};
        llg_rhs(o, St, B, f);
        const double q0 = o.sx[l] + 0.5 * o.dt * (k1[3 * l] + f[0]);
        const double q1 = o.sy[l] + 0.5 * o.dt * (k1[3 * l + 1] + f[1]);
        const double q2 = o.sz[l] + 0.5 * o.dt * (k1[3 * l + 2] + f[2]);
        const double nrm = std::sqrt(q0 * q0 + q1 * q1 + q2 * q2);
        n0[l] = q0 / nrm; n1[l] = q1 / nrm; n2[l] = q2 / nrm;
      }
  o.sx.swap(n0); o.sy.swap(n1); o.sz.swap(n2);
  o.step += 1;
}

// Incoming-slab seeding for one magnetic site (S:S3).  v = track mean spin of the site's
// macrocell, m = min(1,|v|), n^ = v/|v| (z^ if v = 0), theta = theta_max(m) u0, phi = 2 pi u1
// (Philox stream 1, counter n := pass), S = sin(theta)cos(phi) e1 + sin(theta)sin(phi) e2 + cos(theta) n^,
// e1 = normalise(n^ x x^) (n^ x y^ if |n^_x| > 0.9), e2 = n^ x e1.
void seed_site_about(const Oracle& o, int64_t gx, int k, int j, const double v[3], double S[3]);
void seed_site(const Oracle& o, int64_t gx, int k, int j, double S[3]) {
  const int64_t c = o.cell_of(gx, j, k);
  seed_site_about(o, gx, k, j, &o.init_mean[3 * c], S);
}
// v = M / M_S^0 of the cell the site is generated from (track cell, or micromagnetic cell: m_e(T) m)
void seed_site_about(const Oracle& o, int64_t gx, int k, int j, const double v[3], double S[3]) {
  const double v0 = v[0], v1 = v[1], v2 = v[2];
  const double vn = std::sqrt(v0 * v0 + v1 * v1 + v2 * v2);
  const double m = std::fmin(1.0, vn);
  double n[3] = {0.0, 0.0, 1.0};
  if (vn > 0.0) { n[0] = v0 / vn; n[1] = v1 / vn; n[2] = v2 / vn; }
  double e1[3];
  if (std::fabs(n[0]) > 0.9) {  // n x y^ = (-n_z, 0, n_x)
    e1[0] = -n[2]; e1[1] = 0.0; e1[2] = n[0];
  } else {                      // n x x^ = (0, n_z, -n_y)
    e1[0] = 0.0; e1[1] = n[2]; e1[2] = -n[1];
  }
  const double e1n = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
  e1[0] /= e1n; e1[1] /= e1n; e1[2] /= e1n;
  const double e2[3] = {n[1] * e1[2] - n[2] * e1[1], n[2] * e1[0] - n[0] * e1[2],
                        n[0] * e1[1] - n[1] * e1[0]};
  uint32_t r[4];
  const uint64_t g = (uint64_t)((gx * o.nz + k) * o.ny + j);
  philox_block(o.seed, (uint64_t)o.pass, g, 1u, r);
  const double theta = theta_max_of_m(m) * uniform_from_u32(r[0]);
  const double phi = 2.0 * kPi * uniform_from_u32(r[1]);
  const double st = std::sin(theta), ct = std::cos(theta), cp = std::cos(phi), sp = std::sin(phi);
  for (int a = 0; a < 3; ++a) S[a] = st * cp * e1[a] + st * sp * e2[a] + ct * n[a];
}

// ============================================================================================================
// Multiscale window: micromagnetic LLG meshes (S:8(f) item 3).  Readings M1-M10 of DESIGN.md sec. 14.
// ============================================================================================================
// Langevin function B(x) = coth(x) - 1/x, with its series where the difference cancels.
double langevin(double x) {
  if (std::fabs(x) < 1e-3) return x / 3.0 - x * x * x / 45.0 + 2.0 * x * x * x * x * x / 945.0;
  return 1.0 / std::tanh(x) - 1.0 / x;
}
// Equilibrium magnetisation scaling m_e(T) = B[m_e 3 T_C / T + mu_S B_ext / (k_B T)]  (B_ext = mu_0 H_ext, Tesla):
// the largest root in [0, 1].  g(m) = B(beta m + h) - m is concave on m > 0 with g(1) < 0, so that root is unique
// whenever g is positive just above 0 (h > 0, or h = 0 and T < T_C); otherwise m_e = 0.
double m_e_of(double T, double Tc, double mu_s_Bext) {
  if (!(T > 0.0)) return 1.0;
  const double beta = 3.0 * Tc / T, h = mu_s_Bext / (kBoltzmann * T);
  double lo = (h > 0.0) ? 0.0 : 1e-9, hi = 1.0;
  if (!(langevin(beta * lo + h) - lo > 0.0)) return 0.0;
  for (int it = 0; it < 200; ++it) {
    const double mid = 0.5 * (lo + hi);
    if (langevin(beta * mid + h) - mid > 0.0) lo = mid; else hi = mid;
  }
  return 0.5 * (lo + hi);
}

inline int64_t mm_cx0(const Oracle& o, int side) {              // global x index of the mesh's first cell column
  return side == 0 ? o.x0 / o.macro[0] - o.mesh[0].mcx : (o.x0 + o.nx) / o.macro[0];
}
inline size_t mm_idx(const Oracle& o, int a, int b, int c) { return ((size_t)a * o.ncy + b) * o.ncz + c; }
inline int32_t mm_grain_of(const Oracle& o, int64_t cx, int b) {
  if (cx < 0 || cx >= o.ncx || b < 0 || b >= o.ncy) return -1;
  return o.mm_grain[(size_t)(cx * o.ncy + b)];
}
// direction of the frozen track in cell (cx, b, c): what the window has written there, else what lies ahead
bool track_direction(const Oracle& o, int64_t cx, int b, int c, double n[3]) {
  const size_t t = (size_t)((cx * o.ncy + b) * o.ncz + c);
  const double* v = o.out_cnt[t] > 0 ? &o.out_sum[3 * t] : &o.init_mean[3 * t];
  const double vn = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
  if (!(vn > 0.0)) return false;
  n[0] = v[0] / vn; n[1] = v[1] / vn; n[2] = v[2] / vn;
  return true;
}

// M2, M3: per-cell m_e(T) and alpha(T) = lambda (1 - T / 3 T_C) (held at its T = T_C value above T_C)
void mm_refresh_params(Oracle& o) {
  for (int side = 0; side < 2; ++side) {
    Oracle::MicroMesh& M = o.mesh[side];
    const int64_t cx0 = mm_cx0(o, side);
    for (int a = 0; a < M.mcx; ++a)
      for (int b = 0; b < o.ncy; ++b)
        for (int c = 0; c < o.ncz; ++c) {
          const size_t q = mm_idx(o, a, b, c);
          const int32_t g = mm_grain_of(o, cx0 + a, b);
          if (g < 0) { M.me[q] = 0.0; M.alpha[q] = 0.0; continue; }
          const double Bext = std::fabs(o.scale) * std::sqrt(M.Bx[q] * M.Bx[q] + M.By[q] * M.By[q] + M.Bz[q] * M.Bz[q]);
          M.me[q] = m_e_of(M.T[q], o.mm_Tc[g], o.mu_s * Bext);
          M.alpha[q] = o.lambda * (1.0 - std::fmin(M.T[q], o.mm_Tc[g]) / (3.0 * o.mm_Tc[g]));
        }
  }
}

// M9: the two-way exchange of boundary data.  mm_avg = direction of the average atomistic spin in the stencil cell next
// to each mesh; mm_ghost = direction of the mesh cells next to the atomistic mesh.
void mm_exchange(Oracle& o) {
  const int mx = o.macro[0], my = o.macro[1], mz = o.macro[2];
  for (int side = 0; side < 2; ++side) {
    const int i_lo = side == 0 ? 0 : o.nx - mx;
    for (int b = 0; b < o.ncy; ++b)
      for (int c = 0; c < o.ncz; ++c) {
        double s0 = 0, s1 = 0, s2 = 0;
        for (int i = i_lo; i < i_lo + mx; ++i)
          for (int k = c * mz; k < std::min((c + 1) * mz, o.nz); ++k)
            for (int j = b * my; j < std::min((b + 1) * my, o.ny); ++j) {
              if (o.grain_of(i, j) < 0) continue;
              const int64_t l = o.site(i, k, j);
              s0 += o.sx[l]; s1 += o.sy[l]; s2 += o.sz[l];
            }
        const double n = std::sqrt(s0 * s0 + s1 * s1 + s2 * s2);
        double* av = &o.mm_avg[side][3 * ((size_t)b * o.ncz + c)];
        av[0] = n > 0.0 ? s0 / n : 0.0; av[1] = n > 0.0 ? s1 / n : 0.0; av[2] = n > 0.0 ? s2 / n : 0.0;
        const Oracle::MicroMesh& M = o.mesh[side];
        const size_t q = mm_idx(o, side == 0 ? M.mcx - 1 : 0, b, c);
        double* gh = &o.mm_ghost[side][3 * ((size_t)b * o.ncz + c)];
        gh[0] = M.m[3 * q]; gh[1] = M.m[3 * q + 1]; gh[2] = M.m[3 * q + 2];
      }
  }
}

// Effective field of mesh cell (a, b, c), Tesla, for mesh configuration X (M4-M6):
//   B = (2 A(T) / M_S(T)) lap(m) + (2 K(T) / M_S(T)) (m.e) e + s B_app         Eq. (4), (5) in Tesla
//   A(T) = A_0 m_e^2, K(T) = K_0 m_e^3, M_S(T) = M_S^0 m_e  =>  2 A_0 m_e / M_S^0  and  2 K_0 m_e^2 / M_S^0
//   lap(m) by the 6-neighbour stencil: sum over existing neighbours n of the same grain of (m_n - m) / d_n^2.
// A neighbour beyond the mesh is the stencil cell of the atomistic mesh (its average spin direction) on one
// side and the frozen track cell on the other ("the ends of the simulation window are exchange coupled to the track").
void mm_field(const Oracle& o, int side, const std::vector<double>& X, int a, int b, int c, double B[3]) {
  const Oracle::MicroMesh& M = o.mesh[side];
  const size_t q = mm_idx(o, a, b, c);
  const int64_t cx0 = mm_cx0(o, side);
  const int32_t g = mm_grain_of(o, cx0 + a, b);
  B[0] = B[1] = B[2] = 0.0;
  if (g < 0 || !(M.me[q] > 0.0)) return;
  const double m[3] = {X[3 * q], X[3 * q + 1], X[3 * q + 2]};
  auto add = [&](const double* n, int axis) {
    const double pref = 2.0 * o.mm_A0[axis] * M.me[q] / o.mm_Ms0, d = o.mm_cell[axis];
    for (int t = 0; t < 3; ++t) B[t] += pref * (n[t] - m[t]) / (d * d);
  };
  // x neighbours
  for (int dir = -1; dir <= 1; dir += 2) {
    const int a2 = a + dir;
    if (mm_grain_of(o, cx0 + a2, b) != g) continue;
    if (a2 >= 0 && a2 < M.mcx) { add(&X[3 * mm_idx(o, a2, b, c)], 0); continue; }
    const bool towards_atoms = (side == 0) == (dir > 0);
    if (towards_atoms) {
      const double* av = &o.mm_avg[side][3 * ((size_t)b * o.ncz + c)];
      if (av[0] != 0.0 || av[1] != 0.0 || av[2] != 0.0) add(av, 0);
    } else {
      double n[3];
      if (track_direction(o, cx0 + a2, b, c, n)) add(n, 0);
    }
  }
  for (int dir = -1; dir <= 1; dir += 2) {          // y neighbours: the next cell column across the track
    const int b2 = b + dir;
    if (b2 < 0 || b2 >= o.ncy || mm_grain_of(o, cx0 + a, b2) != g) continue;
    add(&X[3 * mm_idx(o, a, b2, c)], 1);
  }
  for (int dir = -1; dir <= 1; dir += 2) {          // z neighbours: same column, same grain
    const int c2 = c + dir;
    if (c2 < 0 || c2 >= o.ncz) continue;
    add(&X[3 * mm_idx(o, a, b, c2)], 2);
  }
  const double* e = &o.axis[3 * g];
  const double ca = 2.0 * o.mm_K0[g] * M.me[q] * M.me[q] / o.mm_Ms0 * (m[0] * e[0] + m[1] * e[1] + m[2] * e[2]);
  for (int t = 0; t < 3; ++t) B[t] += ca * e[t];
  B[0] += o.scale * M.Bx[q]; B[1] += o.scale * M.By[q]; B[2] += o.scale * M.Bz[q];
}

// dm/dt of every cell of one mesh: Eq. (1) without the stochastic field, damping alpha(T), LL form as llg_rhs.
void mm_rhs(const Oracle& o, int side, const std::vector<double>& X, std::vector<double>& f) {
  const Oracle::MicroMesh& M = o.mesh[side];
  f.assign(X.size(), 0.0);
  for (int a = 0; a < M.mcx; ++a)
    for (int b = 0; b < o.ncy; ++b)
      for (int c = 0; c < o.ncz; ++c) {
        const size_t q = mm_idx(o, a, b, c);
        double B[3];
        mm_field(o, side, X, a, b, c, B);
        const double* S = &X[3 * q];
        const double a0 = S[1] * B[2] - S[2] * B[1], a1 = S[2] * B[0] - S[0] * B[2], a2 = S[0] * B[1] - S[1] * B[0];
        const double b0 = S[1] * a2 - S[2] * a1, b1 = S[2] * a0 - S[0] * a2, b2 = S[0] * a1 - S[1] * a0;
        const double al = M.alpha[q], cf = -o.gamma / (1.0 + al * al);
        f[3 * q] = cf * (a0 + al * b0); f[3 * q + 1] = cf * (a1 + al * b1); f[3 * q + 2] = cf * (a2 + al * b2);
      }
}

// M7: one classical RK4 step of length h on both meshes, boundary data held; |m| = 1 restored after the step.
void mm_rk4_step(Oracle& o, double h) {
  for (int side = 0; side < 2; ++side) {
    std::vector<double>& m = o.mesh[side].m;
    std::vector<double> k1, k2, k3, k4, y(m.size());
    mm_rhs(o, side, m, k1);
    for (size_t t = 0; t < m.size(); ++t) y[t] = m[t] + 0.5 * h * k1[t];
    mm_rhs(o, side, y, k2);
    for (size_t t = 0; t < m.size(); ++t) y[t] = m[t] + 0.5 * h * k2[t];
    mm_rhs(o, side, y, k3);
    for (size_t t = 0; t < m.size(); ++t) y[t] = m[t] + h * k3[t];
    mm_rhs(o, side, y, k4);
    for (size_t q = 0; q < m.size() / 3; ++q) {
      double v[3];
      for (int t = 0; t < 3; ++t)
        v[t] = m[3 * q + t] + h / 6.0 * (k1[3 * q + t] + 2.0 * k2[3 * q + t] + 2.0 * k3[3 * q + t] + k4[3 * q + t]);
      const double n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
      for (int t = 0; t < 3; ++t) m[3 * q + t] = n > 0.0 ? v[t] / n : 0.0;
    }
  }
}

// M9: called at the top of every Heun step.  Every mm_every-th step the meshes trade boundary data with the atomistic
// mesh (both directions, from the configurations at that instant) and advance by one RK4 step of mm_every * dt; the
// atomistic mesh then takes its mm_every Heun steps against the held mesh directions.
void mm_before_heun_step(Oracle& o) {
  if (!o.mm) return;
  if (o.mm_age % o.mm_every == 0) {
    mm_exchange(o);
    mm_refresh_params(o);
    mm_rk4_step(o, o.mm_every * o.dt);
  }
  o.mm_age += 1;
}

// number of magnetic sites of track cell (cx, b, c)
int64_t cell_site_count(const Oracle& o, int64_t cx, int b, int c) {
  int64_t n = 0;
  for (int64_t gx = cx * o.macro[0]; gx < std::min<int64_t>((cx + 1) * o.macro[0], o.track_nx); ++gx)
    for (int j = b * o.macro[1]; j < std::min((b + 1) * o.macro[1], o.ny); ++j)
      if (o.grain_map[(size_t)(gx * o.ny + j)] >= 0) n += std::min((c + 1) * o.macro[2], o.nz) - c * o.macro[2];
  return n;
}

// The first `count` cell columns of a mesh go to the track store: M / M_S^0 = m_e m on the magnetic sites of each cell.
void mm_columns_to_track(Oracle& o, int side, int count) {
  const Oracle::MicroMesh& M = o.mesh[side];
  const int64_t cx0 = mm_cx0(o, side);
  for (int a = 0; a < count; ++a)
    for (int b = 0; b < o.ncy; ++b)
      for (int c = 0; c < o.ncz; ++c) {
        if (mm_grain_of(o, cx0 + a, b) < 0) continue;
        const size_t q = mm_idx(o, a, b, c);
        const size_t t = (size_t)(((cx0 + a) * o.ncy + b) * o.ncz + c);
        const int64_t n = cell_site_count(o, cx0 + a, b, c);
        for (int u = 0; u < 3; ++u) o.out_sum[3 * t + u] += M.me[q] * M.m[3 * q + u] * (double)n;
        o.out_cnt[t] += n;
      }
}

// Mesh state = the direction of the track the meshes lie over (empty cells 0): at enable time and at the start of a pass.
void mm_init_from_track(Oracle& o) {
  for (int side = 0; side < 2; ++side) {
    Oracle::MicroMesh& M = o.mesh[side];
    const int64_t cx0 = mm_cx0(o, side);
    for (int a = 0; a < M.mcx; ++a)
      for (int b = 0; b < o.ncy; ++b)
        for (int c = 0; c < o.ncz; ++c) {
          double n[3] = {0.0, 0.0, 0.0};
          if (mm_grain_of(o, cx0 + a, b) >= 0) {
            n[2] = 1.0;
            track_direction(o, cx0 + a, b, c, n);
          }
          for (int u = 0; u < 3; ++u) M.m[3 * mm_idx(o, a, b, c) + u] = n[u];
        }
  }
}

// M10: the window moves by pc whole cells ("in steps set by the track discretization cellsize").
//   trailing mesh -> track (as M / M_S^0 = m_e m on the cell's magnetic sites);  outgoing atomistic planes -> the
//   trailing mesh by Eq. (6) ("averaging", Fig. 1);  incoming atomistic planes <- the leading mesh by the cone
//   thermalisation about m with magnitude m_e ("thermalization", Fig. 1);  leading mesh <- the track ahead.
void seed_plane_from(Oracle& o, int i, int64_t gx, const Oracle::MicroMesh* from, int a_from);
int mm_shift(Oracle& o, int p) {
  const int mx = o.macro[0];
  if (p % mx != 0) return 1;
  const int pc = p / mx;
  Oracle::MicroMesh &L = o.mesh[0], &R = o.mesh[1];
  if (pc > L.mcx || pc > R.mcx) return 1;
  if (mm_cx0(o, 1) + R.mcx + pc > o.ncx) return 1;
  const int64_t cxL = mm_cx0(o, 0), cxA = o.x0 / mx, cxR = mm_cx0(o, 1);
  // 1. trailing mesh columns a < pc -> track
  mm_columns_to_track(o, 0, pc);
  // 2. trailing mesh moves; its new columns are the Eq. (6) averages of the outgoing atomistic cells (direction)
  std::vector<double> newL((size_t)pc * o.ncy * o.ncz * 3, 0.0);
  for (int a = 0; a < pc; ++a)
    for (int b = 0; b < o.ncy; ++b)
      for (int c = 0; c < o.ncz; ++c) {
        if (mm_grain_of(o, cxA + a, b) < 0) continue;
        double s[3] = {0, 0, 0};
        for (int i = a * mx; i < (a + 1) * mx; ++i)
          for (int k = c * o.macro[2]; k < std::min((c + 1) * o.macro[2], o.nz); ++k)
            for (int j = b * o.macro[1]; j < std::min((b + 1) * o.macro[1], o.ny); ++j) {
              if (o.grain_of(i, j) < 0) continue;
              const int64_t l = o.site(i, k, j);
              s[0] += o.sx[l]; s[1] += o.sy[l]; s[2] += o.sz[l];
            }
        const double n = std::sqrt(s[0] * s[0] + s[1] * s[1] + s[2] * s[2]);
        double* d = &newL[3 * mm_idx(o, a, b, c)];
        if (n > 0.0) { d[0] = s[0] / n; d[1] = s[1] / n; d[2] = s[2] / n; } else { d[2] = 1.0; }
      }
  const size_t col = (size_t)o.ncy * o.ncz * 3;
  for (int a = 0; a + pc < L.mcx; ++a) std::memcpy(&L.m[a * col], &L.m[(a + pc) * col], sizeof(double) * col);
  for (int a = 0; a < pc; ++a) std::memcpy(&L.m[(L.mcx - pc + a) * col], &newL[a * col], sizeof(double) * col);
  // 3. atomistic planes move; the incoming ones are generated from the leading mesh's first pc columns
  for (int i = 0; i + p < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        const int64_t l = o.site(i, k, j), s = o.site(i + p, k, j);
        o.sx[l] = o.sx[s]; o.sy[l] = o.sy[s]; o.sz[l] = o.sz[s];
      }
  for (int i = o.nx - p; i < o.nx; ++i) seed_plane_from(o, i, o.x0 + p + i, &R, (i - (o.nx - p)) / mx);
  // 4. leading mesh moves; its new columns are the track ahead (direction)
  for (int a = 0; a + pc < R.mcx; ++a) std::memcpy(&R.m[a * col], &R.m[(a + pc) * col], sizeof(double) * col);
  for (int a = 0; a < pc; ++a)
    for (int b = 0; b < o.ncy; ++b)
      for (int c = 0; c < o.ncz; ++c) {
        double* d = &R.m[3 * mm_idx(o, R.mcx - pc + a, b, c)];
        d[0] = d[1] = d[2] = 0.0;
        const int64_t cx = cxR + R.mcx + a;
        if (mm_grain_of(o, cx, b) < 0) continue;
        const double* v = &o.init_mean[3 * (size_t)((cx * o.ncy + b) * o.ncz + c)];
        const double n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        if (n > 0.0) { d[0] = v[0] / n; d[1] = v[1] / n; d[2] = v[2] / n; } else { d[2] = 1.0; }
      }
  o.x0 += p; o.shift += 1;
  o.mm_age = 0; o.demag_age = 0; o.stray_dirty = true;
  return 0;
}

// Window plane i becomes global plane gx, generated from mesh cell column a_from of `from` (v = m_e m).
void seed_plane_from(Oracle& o, int i, int64_t gx, const Oracle::MicroMesh* from, int a_from) {
  for (int k = 0; k < o.nz; ++k)
    for (int j = 0; j < o.ny; ++j) {
      const int64_t l = o.site(i, k, j);
      if (o.grain_map[(size_t)(gx * o.ny + j)] < 0) { o.sx[l] = o.sy[l] = o.sz[l] = 0.0; continue; }
      const size_t q = mm_idx(o, a_from, j / o.macro[1], k / o.macro[2]);
      const double v[3] = {from->me[q] * from->m[3 * q], from->me[q] * from->m[3 * q + 1], from->me[q] * from->m[3 * q + 2]};
      double S[3];
      seed_site_about(o, gx, k, j, v, S);
      o.sx[l] = S[0]; o.sy[l] = S[1]; o.sz[l] = S[2];
    }
}

// Window plane i becomes global plane gx of the track: vacant columns 0, magnetic sites seeded (S3).
void seed_plane(Oracle& o, int i, int64_t gx) {
  for (int k = 0; k < o.nz; ++k)
    for (int j = 0; j < o.ny; ++j) {
      const int64_t l = o.site(i, k, j);
      if (o.grain_map[(size_t)(gx * o.ny + j)] < 0) { o.sx[l] = o.sy[l] = o.sz[l] = 0.0; continue; }
      double S[3];
      seed_site(o, gx, k, j, S);
      o.sx[l] = S[0]; o.sy[l] = S[1]; o.sz[l] = S[2];
    }
}

}  // namespace

// ============================================================================
// C interface for ctypes (oracle/asd_oracle.py).  Its own description struct: nothing here is
// shared with include/asd.h.
// ============================================================================
extern "C" {

struct orc_desc {
  int32_t lattice, nx, ny, nz;
  int32_t pbc[3];
  int32_t n_grains;
  double mu_s, lambda, gamma, dt;
  double J[3];
  int64_t track_nx, x0;
  const int32_t* grain_map;   // [track_nx*ny]
  const double* grain_ku;     // [n_grains]
  const double* grain_axis;   // [n_grains*3]
  int32_t macro[3];
  int32_t ell_width;
  const int32_t* ell_idx;     // [N*ell_width] or null
  const double* ell_J;        // [N*ell_width] or null
  uint64_t seed;
};

void* orc_create(const orc_desc* d) {
  if (!d || d->nx < 1 || d->ny < 1 || d->nz < 1) return nullptr;
  for (int a = 0; a < 3; ++a) {
    const int n = (a == 0) ? d->nx : (a == 1 ? d->ny : d->nz);
    if (d->pbc[a] && n < 3) return nullptr;  // S:Q17
  }
  if (d->track_nx < d->x0 + d->nx || d->x0 < 0) return nullptr;
  Oracle* o = new Oracle();
  o->lattice = d->lattice; o->nx = d->nx; o->ny = d->ny; o->nz = d->nz;
  for (int a = 0; a < 3; ++a) { o->pbc[a] = d->pbc[a]; o->J[a] = d->J[a]; o->macro[a] = d->macro[a] > 0 ? d->macro[a] : 1; }
  o->mu_s = d->mu_s; o->lambda = d->lambda; o->gamma = d->gamma; o->dt = d->dt;
  o->track_nx = d->track_nx; o->x0 = d->x0; o->n_grains = d->n_grains; o->seed = d->seed;
  o->grain_map.assign(d->grain_map, d->grain_map + (size_t)(d->track_nx * d->ny));
  o->ku.assign(d->grain_ku, d->grain_ku + d->n_grains);
  o->axis.assign(d->grain_axis, d->grain_axis + 3 * (size_t)d->n_grains);
  o->N = (int64_t)d->nx * d->ny * d->nz;
  if (d->ell_width > 0 && d->ell_idx && d->ell_J) {
    o->ell_width = d->ell_width;
    o->ell_idx.assign(d->ell_idx, d->ell_idx + (size_t)(o->N * d->ell_width));
    o->ell_J.assign(d->ell_J, d->ell_J + (size_t)(o->N * d->ell_width));
  }
  const size_t N = (size_t)o->N;
  o->sx.assign(N, 0.0); o->sy.assign(N, 0.0); o->sz.assign(N, 0.0);
  o->T.assign(N, 0.0); o->Bx.assign(N, 0.0); o->By.assign(N, 0.0); o->Bz.assign(N, 0.0);
  o->ncx = (o->track_nx + o->macro[0] - 1) / o->macro[0];
  o->ncy = (o->ny + o->macro[1] - 1) / o->macro[1];
  o->ncz = (o->nz + o->macro[2] - 1) / o->macro[2];
  const size_t nc = (size_t)(o->ncx * o->ncy * o->ncz);
  o->out_sum.assign(3 * nc, 0.0); o->out_cnt.assign(nc, 0);
  o->init_mean.assign(3 * nc, 0.0);
  for (size_t c = 0; c < nc; ++c) o->init_mean[3 * c + 2] = 1.0;  // default track state +z, m0 = 1
  return o;
}

void orc_destroy(void* h) { delete static_cast<Oracle*>(h); }

void orc_set_threads(void* h, int n) {
  static_cast<Oracle*>(h)->threads = n;   // 0 = automatic (see thread_count)
}

int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// fp32 inputs (the same arrays the GPU gets), widened without renormalising (S:O1); vacant -> 0.
void orc_set_spins(void* h, const float* sx, const float* sy, const float* sz) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.demag_age = 0;
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        const int64_t l = o.site(i, k, j);
        const bool mag = o.grain_of(i, j) >= 0;
        o.sx[l] = mag ? (double)sx[l] : 0.0;
        o.sy[l] = mag ? (double)sy[l] : 0.0;
        o.sz[l] = mag ? (double)sz[l] : 0.0;
      }
}

// fp64 spins as they are (vacant -> 0): for harnesses that move planes between oracles (slab decomposition tests).
void orc_set_spins_f64(void* h, const double* sx, const double* sy, const double* sz) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.demag_age = 0; o.mm_age = 0;
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        const int64_t l = o.site(i, k, j);
        const bool mag = o.grain_of(i, j) >= 0;
        o.sx[l] = mag ? sx[l] : 0.0; o.sy[l] = mag ? sy[l] : 0.0; o.sz[l] = mag ? sz[l] : 0.0;
      }
}

void orc_get_spins(void* h, double* sx, double* sy, double* sz) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(sx, o.sx.data(), sizeof(double) * (size_t)o.N);
  std::memcpy(sy, o.sy.data(), sizeof(double) * (size_t)o.N);
  std::memcpy(sz, o.sz.data(), sizeof(double) * (size_t)o.N);
}

void orc_set_fields(void* h, const float* T, const float* Bx, const float* By, const float* Bz) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int64_t l = 0; l < o.N; ++l) {
    if (T) o.T[l] = (double)T[l];
    if (Bx) o.Bx[l] = (double)Bx[l];
    if (By) o.By[l] = (double)By[l];
    if (Bz) o.Bz[l] = (double)Bz[l];
  }
}

// Switches the demagnetising field on: spacing = lattice constants (ax, ay, az) in metres; cell = macro * spacing.
void orc_enable_demag(void* h, const double spacing[3]) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int a = 0; a < 3; ++a) o.cell_m[a] = o.macro[a] * spacing[a];
  o.dcx = (o.nx + o.macro[0] - 2) / o.macro[0] + 1;     // cells overlapped at the worst alignment of x0
  o.dcy = (o.ny + o.macro[1] - 1) / o.macro[1];
  o.dcz = (o.nz + o.macro[2] - 1) / o.macro[2];
  const int sx = 2 * o.dcx - 1, sy = 2 * o.dcy - 1, sz = 2 * o.dcz - 1;
  o.demag_N.assign((size_t)sx * sy * sz * 6, 0.0);
  for (int a = 0; a < sx; ++a)
    for (int b = 0; b < sy; ++b)
      for (int c = 0; c < sz; ++c) {
        const double R[3] = {(a - o.dcx + 1) * o.cell_m[0], (b - o.dcy + 1) * o.cell_m[1], (c - o.dcz + 1) * o.cell_m[2]};
        newell_tensor(o.cell_m, R, &o.demag_N[(((size_t)a * sy + b) * sz + c) * 6]);
      }
  o.demag = true;
  o.demag_age = 0; o.stray_dirty = true;
}
void orc_set_demag_every(void* h, int every) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.demag_every = every; o.demag_age = 0;
}
void orc_newell_tensor(const double cell[3], const double R[3], double out[6]) { newell_tensor(cell, R, out); }
// Demagnetising field of the current spins per window macrocell, Tesla: out[dcx*dcy*dcz*3]; dims returned.
void orc_demag_cells(void* h, double* out, int64_t dims[3]) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::vector<double> Bd;
  demag_cells(o, o.sx.data(), o.sy.data(), o.sz.data(), Bd);
  dims[0] = o.dcx; dims[1] = o.dcy; dims[2] = o.dcz;
  if (out) for (size_t t = 0; t < Bd.size(); ++t) out[t] = Bd[t];
}

// Stray field of the frozen track (reading D4) on / off; range_cells = 0: every track cell is a source.  Needs the
// demagnetising field (its cell geometry).  Returns 0, or 4 if orc_enable_demag has not been called.
int orc_enable_track_stray(void* h, int on, int range_cells) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!o.demag) return 4;
  o.stray = on != 0; o.stray_range = range_cells > 0 ? range_cells : 0; o.stray_dirty = true; o.demag_age = 0;
  return 0;
}
// The track's stray field per window macrocell for the current window origin and track state, Tesla: out[dcx*dcy*dcz*3].
void orc_stray_cells(void* h, double* out) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::vector<double> Bs;
  stray_cells(o, Bs);
  for (size_t t = 0; t < Bs.size(); ++t) out[t] = Bs[t];
}

// Window ends exchange coupled to the frozen track (reading E1); superseded by the meshes of a multiscale window.
void orc_enable_track_exchange(void* h, int on) { static_cast<Oracle*>(h)->track_exch = on != 0; }

void orc_set_field_scale(void* h, float s) { static_cast<Oracle*>(h)->scale = (double)s; }

void orc_step_heun(void* h, int64_t n) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int64_t s = 0; s < n; ++s) heun_step(o);
}

// Deterministic field (no noise) or field with the noise of the current step counter, Tesla.
void orc_field(void* h, int with_noise, double* bx, double* by, double* bz) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (o.mm) mm_exchange(o);
  std::vector<double> Bd;
  if (o.demag) { demag_cells(o, o.sx.data(), o.sy.data(), o.sz.data(), Bd); add_stray(o, Bd); }
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        const int64_t l = o.site(i, k, j);
        bx[l] = by[l] = bz[l] = 0.0;
        if (o.grain_of(i, j) < 0) continue;
        double xi[3], B[3];
        if (with_noise) normals3(o.seed, (uint64_t)o.step, (uint64_t)(((o.x0 + i) * o.nz + k) * o.ny + j), xi);
        field_at(o, o.sx.data(), o.sy.data(), o.sz.data(), i, k, j, with_noise ? xi : nullptr, B,
                 o.demag ? demag_of_site(o, Bd, i, k, j) : nullptr);
        bx[l] = B[0]; by[l] = B[1]; bz[l] = B[2];
      }
}

// E = -1/2 sum_i sum_{j in N(i)} J_ij S_i.S_j - sum_i k_u,g (S_i.e_g)^2 - mu_s sum_i s B_app,i.S_i
// (each bond once; the convention under which Eq. (8) gives T_C = eps z J / 3 k_B; S:O3).
double orc_energy(void* h) {
  Oracle& o = *static_cast<Oracle*>(h);
  double E = 0.0;
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        const int32_t g = o.grain_of(i, j);
        if (g < 0) continue;
        const int64_t l = o.site(i, k, j);
        double e[3];
        exchange_sum(o, o.sx.data(), o.sy.data(), o.sz.data(), i, k, j, e);
        E -= 0.5 * (o.sx[l] * e[0] + o.sy[l] * e[1] + o.sz[l] * e[2]);
        const double d = o.sx[l] * o.axis[3 * g] + o.sy[l] * o.axis[3 * g + 1] + o.sz[l] * o.axis[3 * g + 2];
        E -= o.ku[g] * d * d;
        E -= o.mu_s * o.scale * (o.Bx[l] * o.sx[l] + o.By[l] * o.sy[l] + o.Bz[l] * o.sz[l]);
      }
  return E;
}

// m = sum_{magnetic i} S_i / N_mag  (Eq. (6) with V = whole window; S:O6).
void orc_magnetisation(void* h, double m[3], double* n_magnetic) {
  Oracle& o = *static_cast<Oracle*>(h);
  double s0 = 0, s1 = 0, s2 = 0; int64_t cnt = 0;
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        if (o.grain_of(i, j) < 0) continue;
        const int64_t l = o.site(i, k, j);
        s0 += o.sx[l]; s1 += o.sy[l]; s2 += o.sz[l]; ++cnt;
      }
  const double inv = cnt > 0 ? 1.0 / (double)cnt : 0.0;
  m[0] = s0 * inv; m[1] = s1 * inv; m[2] = s2 * inv;
  if (n_magnetic) *n_magnetic = (double)cnt;
}

void orc_grain_magnetisation(void* h, double* m /* [n_grains*3] */) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::vector<double> s(3 * (size_t)o.n_grains, 0.0); std::vector<int64_t> c((size_t)o.n_grains, 0);
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        const int32_t g = o.grain_of(i, j);
        if (g < 0) continue;
        const int64_t l = o.site(i, k, j);
        s[3 * g] += o.sx[l]; s[3 * g + 1] += o.sy[l]; s[3 * g + 2] += o.sz[l]; ++c[g];
      }
  for (int g = 0; g < o.n_grains; ++g)
    for (int a = 0; a < 3; ++a) m[3 * g + a] = c[g] > 0 ? s[3 * g + a] / (double)c[g] : 0.0;
}

// Window shift by p planes (S:O5).
int orc_shift_window(void* h, int32_t p) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (p < 1 || p > o.nx) return 1;
  if (o.ell_width > 0) return 5;                       // general ELL cannot follow the window
  if (o.x0 + p + o.nx > o.track_nx) return 1;          // grain map must cover the new window
  if (o.mm) return mm_shift(o, p);                     // multiscale window: whole cells, through the meshes (M10)
  o.demag_age = 0;                                     // a held demagnetising field belongs to the old window
  const int nx = o.nx, ny = o.ny, nz = o.nz;
  // S2 outgoing: planes i < p, magnetic sites only, ascending l.
  for (int i = 0; i < p; ++i)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j) {
        if (o.grain_of(i, j) < 0) continue;
        const int64_t l = o.site(i, k, j);
        const int64_t c = o.cell_of(o.x0 + i, j, k);
        o.out_sum[3 * c] += o.sx[l]; o.out_sum[3 * c + 1] += o.sy[l]; o.out_sum[3 * c + 2] += o.sz[l];
        o.out_cnt[c] += 1;
      }
  // move: S(i,.,.) <- S(i+p,.,.) for i < nx-p
  for (int i = 0; i + p < nx; ++i)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j) {
        const int64_t l = o.site(i, k, j), s = o.site(i + p, k, j);
        o.sx[l] = o.sx[s]; o.sy[l] = o.sy[s]; o.sz[l] = o.sz[s];
      }
  // S3 incoming: planes i >= nx-p; new global plane gx = x0 + p + i.
  for (int i = nx - p; i < nx; ++i) seed_plane(o, i, o.x0 + p + i);
  o.x0 += p; o.shift += 1;                              // S4: T and B are NOT moved
  o.stray_dirty = true;
  return 0;
}

// ---- Passes over the track (S:8(f) item 4; sec. III / Fig. 4: "The two tracks were written sequentially ...
// The written bit pattern was then used as the starting state for a second pass through the track shifting algorithm").
// Readings T1-T3 of DESIGN.md sec. 13.
//
// T1 end of a pass: the planes still inside the window are transferred to the track by Eq. (6) exactly as outgoing
//    planes are (S2), and every macrocell the pass has written (count > 0) becomes what lies ahead of the next pass:
//    init_mean[c] = out_sum[c] / out_cnt[c]  (mean spin = M / M_S^0 of the cell).  Cells never written keep their value.
//    The written store is kept (orc_track_get / orc_track_read_scan read it).
//    Multiscale window (reading T1'): the cells of both meshes go to the track as well, as m_e m on their magnetic
//    sites -- exactly what a shift does with the trailing mesh's outgoing columns (M10).
int orc_track_end_pass(void* h) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (o.ell_width > 0) return 5;
  if (o.mm) { mm_columns_to_track(o, 0, o.mesh[0].mcx); mm_columns_to_track(o, 1, o.mesh[1].mcx); }
  for (int i = 0; i < o.nx; ++i)
    for (int k = 0; k < o.nz; ++k)
      for (int j = 0; j < o.ny; ++j) {
        if (o.grain_of(i, j) < 0) continue;
        const int64_t l = o.site(i, k, j);
        const int64_t c = o.cell_of(o.x0 + i, j, k);
        o.out_sum[3 * c] += o.sx[l]; o.out_sum[3 * c + 1] += o.sy[l]; o.out_sum[3 * c + 2] += o.sz[l];
        o.out_cnt[c] += 1;
      }
  const size_t nc = (size_t)(o.ncx * o.ncy * o.ncz);
  for (size_t c = 0; c < nc; ++c) {
    if (o.out_cnt[c] == 0) continue;
    for (int a = 0; a < 3; ++a) o.init_mean[3 * c + a] = o.out_sum[3 * c + a] / (double)o.out_cnt[c];
  }
  o.stray_dirty = true; o.demag_age = 0;
  return 0;
}

// T2 start of the next pass: the written store is cleared, pass += 1, the window returns to global plane x0_new and
//    ALL its planes are generated from the track by the cone thermalisation of P:68 (S3), Philox counter n := pass.
//    The step and shift counters run on.
//    Multiscale window (reading T2'): x0_new must be a whole number of cells with both meshes inside the track; the
//    meshes restart from the direction of the track they now lie over, as at enable time.
int orc_track_begin_pass(void* h, int64_t x0_new) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (o.ell_width > 0) return 5;
  if (x0_new < 0 || x0_new + o.nx > o.track_nx) return 1;
  if (o.mm && (x0_new % o.macro[0] != 0 || x0_new / o.macro[0] - o.mesh[0].mcx < 0 ||
               (x0_new + o.nx) / o.macro[0] + o.mesh[1].mcx > o.ncx)) return 1;
  const size_t nc = (size_t)(o.ncx * o.ncy * o.ncz);
  for (size_t c = 0; c < nc; ++c) { o.out_cnt[c] = 0; o.out_sum[3 * c] = o.out_sum[3 * c + 1] = o.out_sum[3 * c + 2] = 0.0; }
  o.pass += 1;
  o.x0 = x0_new;
  o.demag_age = 0; o.stray_dirty = true;
  for (int i = 0; i < o.nx; ++i) seed_plane(o, i, o.x0 + i);
  if (o.mm) { mm_init_from_track(o); o.mm_age = 0; mm_refresh_params(o); }
  return 0;
}

// T3 read-back figure of merit, standing in for the TMR read head of P:114 (which needs a solver that is not part of
//    the method): the mean S_z per magnetic site under a Gaussian reader footprint, from the WRITTEN store,
//      R(x_r) = sum_c w_c sum_z[c] / sum_c w_c cnt[c],   w_c = exp(-(x_c - x_r)^2 / (2 sx^2) - (y_c - y_r)^2 / (2 sy^2)),
//    (x_c, y_c) = nominal centre of macrocell c in site units ((cx + 1/2) mx, (cy + 1/2) my), all layers cz summed;
//    x_r = x_first + n x_step, n = 0..count-1.  0 where the footprint holds no written site.
void orc_track_read_scan(void* h, double y_r, double sigma_x, double sigma_y, double x_first, double x_step,
                         int64_t count, double* out) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int64_t n = 0; n < count; ++n) {
    const double x_r = x_first + (double)n * x_step;
    double num = 0.0, den = 0.0;
    for (int64_t cx = 0; cx < o.ncx; ++cx)
      for (int64_t cy = 0; cy < o.ncy; ++cy) {
        const double xc = ((double)cx + 0.5) * o.macro[0], yc = ((double)cy + 0.5) * o.macro[1];
        const double w = std::exp(-(xc - x_r) * (xc - x_r) / (2.0 * sigma_x * sigma_x)
                                  - (yc - y_r) * (yc - y_r) / (2.0 * sigma_y * sigma_y));
        for (int64_t cz = 0; cz < o.ncz; ++cz) {
          const size_t c = (size_t)((cx * o.ncy + cy) * o.ncz + cz);
          num += w * o.out_sum[3 * c + 2];
          den += w * (double)o.out_cnt[c];
        }
      }
    out[n] = den > 0.0 ? num / den : 0.0;
  }
}

void orc_track_set_init(void* h, const float* mean_spin /* [ncell*3] or null */, float m0) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.stray_dirty = true; o.demag_age = 0;
  const size_t nc = (size_t)(o.ncx * o.ncy * o.ncz);
  for (size_t c = 0; c < nc; ++c)
    for (int a = 0; a < 3; ++a)
      o.init_mean[3 * c + a] = mean_spin ? (double)mean_spin[3 * c + a] : (a == 2 ? (double)m0 : 0.0);
}

int64_t orc_track_ncell(void* h, int64_t dims[3]) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (dims) { dims[0] = o.ncx; dims[1] = o.ncy; dims[2] = o.ncz; }
  return o.ncx * o.ncy * o.ncz;
}

// mean_spin[c] = out_sum[c] / out_cnt[c] (0 if empty), count[c] = out_cnt[c]; sums also returned.
void orc_track_get(void* h, double* mean_spin, int64_t* count, double* sum) {
  Oracle& o = *static_cast<Oracle*>(h);
  const size_t nc = (size_t)(o.ncx * o.ncy * o.ncz);
  for (size_t c = 0; c < nc; ++c) {
    if (count) count[c] = o.out_cnt[c];
    for (int a = 0; a < 3; ++a) {
      if (sum) sum[3 * c + a] = o.out_sum[3 * c + a];
      if (mean_spin) mean_spin[3 * c + a] = o.out_cnt[c] > 0 ? o.out_sum[3 * c + a] / (double)o.out_cnt[c] : 0.0;
    }
  }
}

void orc_get_counters(void* h, int64_t* step, int64_t* shift, int64_t* x0, int64_t* pass) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (step) *step = o.step; if (shift) *shift = o.shift; if (x0) *x0 = o.x0; if (pass) *pass = o.pass;
}

void orc_set_counters(void* h, int64_t step, int64_t shift, int64_t pass) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.step = step; o.shift = shift; o.pass = pass;
}

// ---- multiscale window (S:8(f) item 3) ----
struct orc_mm_desc {
  int32_t mcx[2];             // cells along x of the trailing / leading mesh
  int32_t every;              // Heun steps per RK4 step
  double Ms0, A0[3];          // A/m; J/m along x, y, z
  const double* K0;           // [n_grains] J/m^3
  const double* Tc;           // [n_grains] K
  const int32_t* cell_grain;  // [ncx*ncy] grain id per track cell column, -1 = empty
  double spacing[3];          // lattice constants, metres (cell = macro * spacing)
};
// 0 ok; 1 bad geometry (M1: x0 and nx whole cells; meshes inside the track); 5 unsupported lattice options
int orc_mm_enable(void* h, const orc_mm_desc* d) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (o.ell_width > 0 || o.pbc[0] || o.pbc[1] || o.pbc[2]) return 5;
  const int mx = o.macro[0];
  if (o.x0 % mx != 0 || o.nx % mx != 0 || d->mcx[0] < 1 || d->mcx[1] < 1 || d->every < 1) return 1;
  if (o.x0 / mx - d->mcx[0] < 0 || (o.x0 + o.nx) / mx + d->mcx[1] > o.ncx) return 1;
  o.mm_Ms0 = d->Ms0; for (int a = 0; a < 3; ++a) o.mm_A0[a] = d->A0[a]; o.mm_every = d->every; o.mm_age = 0;
  o.mm_K0.assign(d->K0, d->K0 + o.n_grains); o.mm_Tc.assign(d->Tc, d->Tc + o.n_grains);
  o.mm_grain.assign(d->cell_grain, d->cell_grain + (size_t)(o.ncx * o.ncy));
  for (int a = 0; a < 3; ++a) o.mm_cell[a] = o.macro[a] * d->spacing[a];
  for (int side = 0; side < 2; ++side) {
    Oracle::MicroMesh& M = o.mesh[side];
    M.mcx = d->mcx[side];
    const size_t n = (size_t)M.mcx * o.ncy * o.ncz;
    M.m.assign(3 * n, 0.0); M.T.assign(n, 0.0); M.Bx.assign(n, 0.0); M.By.assign(n, 0.0); M.Bz.assign(n, 0.0);
    M.me.assign(n, 0.0); M.alpha.assign(n, 0.0);
    o.mm_ghost[side].assign((size_t)o.ncy * o.ncz * 3, 0.0);
    o.mm_avg[side].assign((size_t)o.ncy * o.ncz * 3, 0.0);
  }
  o.mm = true;
  mm_init_from_track(o);                                  // initial state: the direction of the track under the meshes
  mm_refresh_params(o);
  return 0;
}
int64_t orc_mm_cells(void* h, int side) {
  Oracle& o = *static_cast<Oracle*>(h);
  return (int64_t)o.mesh[side].mcx * o.ncy * o.ncz;
}
// per cell (a slowest, then b, then c): T [K] and B [Tesla]; NULL keeps the previous array
void orc_mm_set_fields(void* h, int side, const double* T, const double* Bx, const double* By, const double* Bz) {
  Oracle& o = *static_cast<Oracle*>(h);
  Oracle::MicroMesh& M = o.mesh[side];
  for (size_t q = 0; q < M.T.size(); ++q) {
    if (T) M.T[q] = T[q];
    if (Bx) M.Bx[q] = Bx[q];
    if (By) M.By[q] = By[q];
    if (Bz) M.Bz[q] = Bz[q];
  }
  mm_refresh_params(o);
}
// m [cells*3]; set: empty cells stay 0, others are stored as given (unit vectors expected)
void orc_mm_set_m(void* h, int side, const double* m) {
  Oracle& o = *static_cast<Oracle*>(h);
  Oracle::MicroMesh& M = o.mesh[side];
  const int64_t cx0 = mm_cx0(o, side);
  for (int a = 0; a < M.mcx; ++a)
    for (int b = 0; b < o.ncy; ++b)
      for (int c = 0; c < o.ncz; ++c) {
        const size_t q = mm_idx(o, a, b, c);
        const bool full = mm_grain_of(o, cx0 + a, b) >= 0;
        for (int u = 0; u < 3; ++u) M.m[3 * q + u] = full ? m[3 * q + u] : 0.0;
      }
  o.mm_age = 0;
}
void orc_mm_get_m(void* h, int side, double* m) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(m, o.mesh[side].m.data(), sizeof(double) * o.mesh[side].m.size());
}
void orc_mm_get_params(void* h, int side, double* me, double* alpha) {
  Oracle& o = *static_cast<Oracle*>(h);
  mm_refresh_params(o);
  std::memcpy(me, o.mesh[side].me.data(), sizeof(double) * o.mesh[side].me.size());
  std::memcpy(alpha, o.mesh[side].alpha.data(), sizeof(double) * o.mesh[side].alpha.size());
}
// effective field of every cell of one mesh for the current configurations (boundary data exchanged now), Tesla
void orc_mm_field(void* h, int side, double* B) {
  Oracle& o = *static_cast<Oracle*>(h);
  mm_exchange(o);
  mm_refresh_params(o);
  const Oracle::MicroMesh& M = o.mesh[side];
  for (int a = 0; a < M.mcx; ++a)
    for (int b = 0; b < o.ncy; ++b)
      for (int c = 0; c < o.ncz; ++c) mm_field(o, side, M.m, a, b, c, &B[3 * mm_idx(o, a, b, c)]);
}
// n RK4 steps of length h on the meshes alone (boundary data exchanged before each): for the pins
void orc_mm_step(void* h, int64_t n, double step) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int64_t t = 0; t < n; ++t) { mm_exchange(o); mm_refresh_params(o); mm_rk4_step(o, step); }
}
double orc_mm_me(double T, double Tc, double mu_s_Bext) { return m_e_of(T, Tc, mu_s_Bext); }
double orc_langevin(double x) { return langevin(x); }

// ---- building blocks exposed for the pins ----
void orc_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) { philox4x32_10(key, ctr, out); }
void orc_philox_block(uint64_t seed, uint64_t n, uint64_t g, uint32_t stream, uint32_t out[4]) { philox_block(seed, n, g, stream, out); }
double orc_uniform(uint32_t r) { return uniform_from_u32(r); }
void orc_normals3(uint64_t seed, uint64_t step, uint64_t g, double xi[3]) { normals3(seed, step, g, xi); }
// Bulk version for moment tests: xi[3*count], sites g0..g0+count-1.
void orc_normals3_bulk(uint64_t seed, uint64_t step, uint64_t g0, int64_t count, double* xi) {
  for (int64_t a = 0; a < count; ++a) normals3(seed, step, g0 + (uint64_t)a, xi + 3 * a);
}
double orc_theta_max(double m) { return theta_max_of_m(m); }
double orc_sigma(void* h, double T) { return sigma_T(*static_cast<Oracle*>(h), T); }

}  // extern "C"
