// oracle/sph_oracle.cpp
//
// TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH.
// Plain, slow, double-precision CPU restatement of the per-time-step particle
// pipeline of arXiv 2110.02621 (Rezavand, Zhang, Hu).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may load this library.  It shares no code, header, table or helper with the
// CUDA path under paper_2110_02621_b200/csrc/.
//
// Every function cites the passage of /root/reference/PAPER.md it follows
// (PAPER.md:<line>, equation number).  Where the paper is silent or garbled the
// reading is the one listed in DESIGN.md ("Readings", ids A1..A28 follow
// SURVEY.md §8(c); A13b, A29-A32 were added by the build).
//
// Pins (tests/test_oracle_pins.py) and what they fix:
//   kernel W, W'          — unit integral, finite difference           (P1)
//   sigma0, W(0)          — lattice constants, partition of unity      (P2)
//   momentum sum          — first-moment lattice constant M1           (P3)
//   wall extrapolation    — exact for a linear hydrostatic field       (P4)
//   neighbour search      — brute force all pairs                      (P6)
//   Riemann terms         — reduction to Eq. 2.5 / 2.6                 (P7)
//   pair force            — antisymmetry m_i a_ij = -m_j a_ji          (P8)
//   continuity            — scalar identity, Galilean invariance       (P9,P10)
//   integrator, dt        — free fall closed form                      (P12)
//   reinitialisation      — Eq. 2.17 cases                             (P13)
//   penalty               — closed form of reading A8/A9               (P15)
//   normals               — flat wall / corner / middle layer          (P16)
//   mass, whole step      — hydrostatic column relaxes to rho g (H-z)  (P5,P17)
//   step dispatch         — which phase gets Eq. 2.17 / 2.18, continuity / summation, whose neighbours
//                           count in sigma: densities after a dt = 0 two-phase step by hand       (P23)
//   stats                 — E_k = 1/2 M |v|^2, mass, x_front closed forms                          (P24)
//   sigma of pass A       — lattice constant after a step                                         (P25)
//   two-phase tank X1     — stays at rest under reading A13b, not without it   (P26)
//   wall extensions       — without them air leaves the tank                   (P27)
//   unequal-c solver      — acoustic characteristic relations, limiter limits                    (P28)
//   fluid-wall pair       — Eq. 2.12 lever, wall density A5, Eq. 2.11 weights by hand             (P29)
// PARITY UNPINNED (fixed by DESIGN.md readings only, no external pin exists):
//   wall velocity mirror (A6), step ordering and two wall passes (A16), penalty scaling and
//   window (A8 / A9); whether A3's extension and A5's per-pair wall density are the authors' choice
//   (P18 / P28 / P29 pin that the code computes what those readings say).
//
// Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py)

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

constexpr int ORC_MAX_PHASES = 4;
constexpr int ORC_TAG_WALL = -1;
constexpr uint32_t ORC_FLAG_REINIT = 1u;
constexpr uint32_t ORC_FLAG_WALL_VEL_MIRROR = 2u;
// NEXT-4 ablation ("compare the results with the method of Adami et al. (2012)"): the wall
// model WITHOUT the paper's extensions: Eq. 2.12 in its single-phase form for every phase (no division by
// rho_f) and no penalty force F_p (Eq. 2.13).
constexpr uint32_t ORC_FLAG_WALL_ADAMI_ONLY = 8u;
// Study-only variants of two readings (NEXT-2, DESIGN.md section 3 A13 / A15); never set by the parity tests:
//   REINIT_LITERAL  the printed assignment of PAPER.md:155: Eq. 2.17 for the light (summation) phases,
//                   Eq. 2.18 for the heavy (continuity) phases, i.e. the reverse of reading A13;
//   SUM_RAW         Eq. 2.4 as printed, rho_i = m_i sum_j W_ij (incl. the self term), instead of the
//                   normalised form rho0 sigma / sigma0 of reading A15.
constexpr uint32_t ORC_VAR_REINIT_LITERAL = 1u;
constexpr uint32_t ORC_VAR_SUM_RAW = 2u;
//   SIGMA_ALL       sigma_i of a free-surface (continuity) phase counts neighbours of EVERY phase, as the
//                   first build of this oracle did; reading A13b counts the particle's own phase and the
//                   walls only (see number density below).
constexpr uint32_t ORC_VAR_SIGMA_ALL = 4u;

struct orc_params {
  int32_t dim;
  int32_t n_phases;
  double dp;
  double h;
  double rho0[ORC_MAX_PHASES];
  double c0[ORC_MAX_PHASES];
  double g[3];
  double g_osc_amp[3];
  double g_osc_period;
  double cfl;
  double penalty_strength;
  uint32_t penalty_phase_mask;
  uint32_t free_surface_mask;
  uint32_t flags;
  uint32_t variant;     // ORC_VAR_* (0 in every parity run)
  double domain_min[3];
  double domain_max[3];
  // NEXT-1: rigid wall motion x_w(t) = x_w(t_start) + A [sin(2 pi f t) - sin(2 pi f t_start)]
  double wall_osc_amp[3];
  double wall_osc_freq;
  double t_start;       // time at orc_set_particles (0 in every BASELINE.json configuration)
};

const double PI = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------
// Smoothing kernel.  PAPER.md:109, :212 "5th-order / quintic Wendland", kappa=2,
// support 2h; formula not printed -> reading A1: Wendland C2
//   W(r) = alpha_d (1 - q/2)^4 (1 + 2q),  q = r/h < 2
//   alpha_2 = 7/(4 pi h^2), alpha_3 = 21/(16 pi h^3)
// ---------------------------------------------------------------------------
double alpha_d(int dim, double h) {
  if (dim == 2) return 7.0 / (4.0 * PI * h * h);
  return 21.0 / (16.0 * PI * h * h * h);
}

double kernel_w(int dim, double h, double r) {
  double q = r / h;
  if (q >= 2.0) return 0.0;
  double t = 1.0 - 0.5 * q;
  return alpha_d(dim, h) * t * t * t * t * (1.0 + 2.0 * q);
}

// dW/dr = -(5 alpha_d / h) q (1 - q/2)^3
double kernel_dw(int dim, double h, double r) {
  double q = r / h;
  if (q >= 2.0) return 0.0;
  double t = 1.0 - 0.5 * q;
  return -5.0 * alpha_d(dim, h) / h * q * t * t * t;
}

// sigma^0: number density of the full undisturbed lattice incl. the self term
// ("initial number particle densities"; reading A12, A14).
double sigma0_lattice(int dim, double h, double dp) {
  int m = (int)std::ceil(2.0 * h / dp) + 1;
  double s = 0.0;
  for (int k = (dim == 3 ? -m : 0); k <= (dim == 3 ? m : 0); ++k)
    for (int j = -m; j <= m; ++j)
      for (int i = -m; i <= m; ++i) {
        double r = dp * std::sqrt((double)(i * i + j * j + k * k));
        s += kernel_w(dim, h, r);
      }
  return s;
}

// ---------------------------------------------------------------------------
// Inter-particle Riemann problem, Eq. 2.7-2.8.
// Equal sound speeds: the paper's formulas literally.
// Unequal sound speeds (BASELINE.json config 2, reading A3): acoustic solver
// with impedances Z = rho c; reduces to Eq. 2.8 at c_L = c_R (pin P18).
// ---------------------------------------------------------------------------
struct Riemann {
  double Ustar, pstar, Ubar;  // Ubar: the average normal velocity removed from v-bar
  double wL, wR;              // weights of v_i, v_j in the averaged velocity of v*
};

Riemann riemann_paper(double rL, double UL, double pL, double rR, double UR, double pR,
                      double c) {
  Riemann s;
  double rbar = 0.5 * (rL + rR);
  s.Ubar = (rL * UL + rR * UR) / (rL + rR);
  double Pbar = (rL * pR + rR * pL) / (rL + rR);
  s.Ustar = s.Ubar + 0.5 * (pL - pR) / (c * rbar);
  double beta = std::min(3.0 * std::max(UL - UR, 0.0), c);
  s.pstar = Pbar + rL * rR * beta * (UL - UR) / (rL + rR);
  s.wL = rL / (rL + rR);
  s.wR = rR / (rL + rR);
  return s;
}

Riemann riemann_acoustic(double rL, double UL, double pL, double cL, double rR, double UR,
                         double pR, double cR) {
  Riemann s;
  double ZL = rL * cL, ZR = rR * cR;
  s.Ubar = (ZL * UL + ZR * UR) / (ZL + ZR);
  s.Ustar = (ZL * UL + ZR * UR + pL - pR) / (ZL + ZR);
  double ctil = (ZL + ZR) / (rL + rR);
  double beta = std::min(3.0 * std::max(UL - UR, 0.0), ctil);
  s.pstar = (ZL * pR + ZR * pL) / (ZL + ZR) + ZL * ZR / (ZL + ZR) * (beta / ctil) * (UL - UR);
  s.wL = ZL / (ZL + ZR);
  s.wR = ZR / (ZL + ZR);
  return s;
}

Riemann riemann(double rL, double UL, double pL, double cL, double rR, double UR, double pR,
                double cR) {
  if (cL == cR) return riemann_paper(rL, UL, pL, rR, UR, pR, cL);
  return riemann_acoustic(rL, UL, pL, cL, rR, UR, pR, cR);
}

// Eq. 2.17 / 2.18.  free_surface != 0 -> Eq. 2.17.
double reinit_density(double rho_star, double rho0, double sigma, double sigma0,
                      int free_surface) {
  double rs = rho0 * sigma / sigma0;
  if (!free_surface) return rs;
  return rs + std::max(0.0, rho_star - rs) * rho0 / rho_star;
}

// ---------------------------------------------------------------------------
struct Ctx {
  orc_params P;
  int64_t n = 0;
  double V0 = 0, sigma0 = 0, t = 0, dt_last = 0;
  int64_t steps = 0, npairs = 0, escaped = 0;
  std::vector<double> r, v, a;          // n*3
  std::vector<double> r0;               // positions at orc_set_particles (wall entries used by the wall motion)
  std::vector<double> rho, p, m, sigma, drho;
  std::vector<int32_t> tag;
  std::vector<double> pw;               // wall pressure (only wall entries used)
  std::vector<double> vw;               // wall velocity for the Riemann problem, n*3
  std::vector<double> nw;               // wall normals, n*3
  // neighbour lists (CSR, j != i, r < 2h, any tag)
  std::vector<int64_t> nb_off;
  std::vector<int32_t> nb;
  int nc[3] = {1, 1, 1};
};

inline bool is_wall(const Ctx& S, int64_t i) { return S.tag[i] == ORC_TAG_WALL; }

void gravity_at(const Ctx& S, double t, double g[3]) {
  for (int k = 0; k < 3; ++k) g[k] = S.P.g[k];
  if (S.P.g_osc_period > 0.0) {
    double s = std::sin(2.0 * PI * t / S.P.g_osc_period);
    for (int k = 0; k < 3; ++k) g[k] += S.P.g_osc_amp[k] * s;
  }
}

// NEXT-1.  Prescribed rigid wall kinematics, "x = A0 sin(2 pi f0 t)": displacement since
// orc_set_particles, wall velocity and wall acceleration a_w (the a_w of Eq. 2.12).
inline bool walls_move(const Ctx& S) {
  return S.P.wall_osc_freq > 0.0 &&
         (S.P.wall_osc_amp[0] != 0.0 || S.P.wall_osc_amp[1] != 0.0 || S.P.wall_osc_amp[2] != 0.0);
}
void wall_motion(const Ctx& S, double t, double s[3], double vwall[3], double aw[3]) {
  for (int k = 0; k < 3; ++k) s[k] = vwall[k] = aw[k] = 0.0;
  if (!walls_move(S)) return;
  const double w = 2.0 * PI * S.P.wall_osc_freq;
  for (int k = 0; k < S.P.dim; ++k) {
    s[k] = S.P.wall_osc_amp[k] * (std::sin(w * t) - std::sin(w * S.P.t_start));
    vwall[k] = S.P.wall_osc_amp[k] * w * std::cos(w * t);
    aw[k] = -S.P.wall_osc_amp[k] * w * w * std::sin(w * t);
  }
}

// Own cell list (double), cell edge 2h, cells clamped to the box (reading A23).
void cell_of(const Ctx& S, const double* x, int c[3]) {
  double L = 2.0 * S.P.h;
  for (int k = 0; k < 3; ++k) {
    if (k >= S.P.dim) { c[k] = 0; continue; }
    int ci = (int)std::floor((x[k] - S.P.domain_min[k]) / L);
    c[k] = std::min(std::max(ci, 0), S.nc[k] - 1);
  }
}

void build_neighbours(Ctx& S) {
  const int64_t n = S.n;
  const double L = 2.0 * S.P.h, rc2 = L * L;
  for (int k = 0; k < 3; ++k)
    S.nc[k] = (k < S.P.dim)
                  ? std::max(1, (int)std::ceil((S.P.domain_max[k] - S.P.domain_min[k]) / L))
                  : 1;
  const int64_t ncell = (int64_t)S.nc[0] * S.nc[1] * S.nc[2];
  std::vector<int64_t> cid(n);
  std::vector<int64_t> start(ncell + 1, 0);
  int64_t esc = 0;
  for (int64_t i = 0; i < n; ++i) {
    int c[3];
    cell_of(S, &S.r[3 * i], c);
    cid[i] = ((int64_t)c[2] * S.nc[1] + c[1]) * S.nc[0] + c[0];
    start[cid[i] + 1]++;
    if (!is_wall(S, i))
      for (int k = 0; k < S.P.dim; ++k)
        if (S.r[3 * i + k] < S.P.domain_min[k] || S.r[3 * i + k] >= S.P.domain_max[k]) {
          esc++;
          break;
        }
  }
  S.escaped = esc;
  for (int64_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
  std::vector<int32_t> order(n);
  {
    std::vector<int64_t> fill(start.begin(), start.end() - 1);
    for (int64_t i = 0; i < n; ++i) order[fill[cid[i]]++] = (int32_t)i;
  }
  std::vector<int64_t> cnt(n + 1, 0);
  std::vector<std::vector<int32_t>> lists(n);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < n; ++i) {
    int c[3];
    cell_of(S, &S.r[3 * i], c);
    std::vector<int32_t>& li = lists[i];
    for (int dz = -1; dz <= 1; ++dz) {
      int z = c[2] + dz;
      if (z < 0 || z >= S.nc[2]) continue;
      for (int dy = -1; dy <= 1; ++dy) {
        int y = c[1] + dy;
        if (y < 0 || y >= S.nc[1]) continue;
        for (int dx = -1; dx <= 1; ++dx) {
          int x = c[0] + dx;
          if (x < 0 || x >= S.nc[0]) continue;
          int64_t cc = ((int64_t)z * S.nc[1] + y) * S.nc[0] + x;
          for (int64_t s = start[cc]; s < start[cc + 1]; ++s) {
            int32_t j = order[s];
            if (j == i) continue;
            double d2 = 0;
            for (int k = 0; k < 3; ++k) {
              double d = S.r[3 * i + k] - S.r[3 * j + k];
              d2 += d * d;
            }
            if (d2 < rc2) li.push_back(j);
          }
        }
      }
    }
    std::sort(li.begin(), li.end());
  }
  S.nb_off.assign(n + 1, 0);
  for (int64_t i = 0; i < n; ++i) S.nb_off[i + 1] = S.nb_off[i] + (int64_t)lists[i].size();
  S.nb.resize(S.nb_off[n]);
  int64_t np = 0;
  for (int64_t i = 0; i < n; ++i) {
    std::copy(lists[i].begin(), lists[i].end(), S.nb.begin() + S.nb_off[i]);
    if (!is_wall(S, i)) np += (int64_t)lists[i].size();
  }
  S.npairs = np;  // directed (i fluid, j any), SURVEY.md §8(c) "Pair counting"
}

// Wall normals, Eq. 2.16; sum over wall particles only.
// Degenerate normals -> 0 (reading A10).
void wall_normals(Ctx& S) {
  const int dim = S.P.dim;
  const double h = S.P.h;
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < S.n; ++i) {
    double psi[3] = {0, 0, 0};
    S.nw[3 * i] = S.nw[3 * i + 1] = S.nw[3 * i + 2] = 0.0;
    if (!is_wall(S, i)) continue;
    for (int64_t s = S.nb_off[i]; s < S.nb_off[i + 1]; ++s) {
      int64_t j = S.nb[s];
      if (!is_wall(S, j)) continue;
      double d[3], r2 = 0;
      for (int k = 0; k < 3; ++k) {
        d[k] = S.r[3 * i + k] - S.r[3 * j + k];
        r2 += d[k] * d[k];
      }
      double r = std::sqrt(r2);
      if (r == 0.0) continue;
      double dw = kernel_dw(dim, h, r);
      for (int k = 0; k < 3; ++k) psi[k] -= S.V0 * dw * d[k] / r;  // -(m_j/rho_j) grad_i W_ij
    }
    double nrm = std::sqrt(psi[0] * psi[0] + psi[1] * psi[1] + psi[2] * psi[2]);
    if (nrm * h >= 1e-3)
      for (int k = 0; k < 3; ++k) S.nw[3 * i + k] = psi[k] / nrm;
  }
}

// Which neighbours j enter sigma_i ("sigma_i = sum W_ij"; reading A13b).  PAPER.md:155: "the
// light phase experiences the heavy phase like moving wall boundary, while the heavy phase undergoes a
// free-surface-like flow with variable free-surface pressure": in a multi-phase run the number density
// of a free-surface (heavy) phase particle counts its own phase and the walls, NOT the light phase, so
// that Eq. 2.17 sees the interface as the free surface the sentence describes; an internal-flow (light)
// phase particle counts every neighbour (the heavy phase is its moving wall).  Single phase: everything.
inline bool counts_in_sigma(const Ctx& S, int64_t i, int64_t j) {
  if (S.P.n_phases < 2 || (S.P.variant & ORC_VAR_SIGMA_ALL) || is_wall(S, i)) return true;
  if (!((S.P.free_surface_mask >> S.tag[i]) & 1u)) return true;
  return is_wall(S, j) || S.tag[j] == S.tag[i];
}

// sigma_i = W(0) + sum_j W_ij (A14, A13b).
void number_density(Ctx& S) {
  const int dim = S.P.dim;
  const double h = S.P.h;
  const double w0 = kernel_w(dim, h, 0.0);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < S.n; ++i) {
    double s = w0;
    for (int64_t q = S.nb_off[i]; q < S.nb_off[i + 1]; ++q) {
      int64_t j = S.nb[q];
      if (!counts_in_sigma(S, i, j)) continue;
      double r2 = 0;
      for (int k = 0; k < 3; ++k) {
        double d = S.r[3 * i + k] - S.r[3 * j + k];
        r2 += d * d;
      }
      s += kernel_w(dim, h, std::sqrt(r2));
    }
    S.sigma[i] = s;
  }
}

// O-1.  PAPER.md:147-159: "At the beginning of every time step, the fluid density
// field is initialised by Eq.(2.17) or Eq.(2.18)"; phase assignment: reading A13.
void reinitialise(Ctx& S) {
  if (!(S.P.flags & ORC_FLAG_REINIT)) return;
  for (int64_t i = 0; i < S.n; ++i) {
    if (is_wall(S, i)) continue;
    int ph = S.tag[i];
    int fs = (S.P.free_surface_mask >> ph) & 1u;
    if (S.P.variant & ORC_VAR_REINIT_LITERAL) fs = !fs;
    S.rho[i] = reinit_density(S.rho[i], S.P.rho0[ph], S.sigma[i], S.sigma0, fs);
    S.p[i] = S.P.c0[ph] * S.P.c0[ph] * (S.rho[i] - S.P.rho0[ph]);  // Eq. 2.3
  }
}

// O-2.  PAPER.md:176-182, Eq. 2.23-2.24; U_max = current max |v| (reading A17).
double time_step(const Ctx& S) {
  double vmax = 0, cmax = 0;
  for (int ph = 0; ph < S.P.n_phases; ++ph) cmax = std::max(cmax, S.P.c0[ph]);
  for (int64_t i = 0; i < S.n; ++i) {
    if (is_wall(S, i)) continue;
    double v2 = 0;
    for (int k = 0; k < 3; ++k) v2 += S.v[3 * i + k] * S.v[3 * i + k];
    vmax = std::max(vmax, std::sqrt(v2));
  }
  double dt = S.P.cfl * S.P.h / (cmax + vmax);
  double g[3];
  gravity_at(S, S.t, g);
  double gn = std::sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
  if (gn > 0.0) dt = std::min(dt, S.P.cfl * std::sqrt(S.P.h / gn));
  return dt;
}

// O-4.  PAPER.md:111-116, Eq. 2.12 (readings A4-A7) at time t: the lever term carries g - a_w(t), the
// mirror 2 v_wall(t) - <v_f> (a_w = 0, v_wall = 0 for the static walls of every BASELINE.json configuration).
void wall_extrapolate(Ctx& S, const double g_in[3], bool with_velocity, double t) {
  double sdis[3], vwall[3], aw[3];
  wall_motion(S, t, sdis, vwall, aw);
  const double g[3] = {g_in[0] - aw[0], g_in[1] - aw[1], g_in[2] - aw[2]};
  const int dim = S.P.dim;
  const double h = S.P.h;
  const bool multi = S.P.n_phases > 1 && !(S.P.flags & ORC_FLAG_WALL_ADAMI_ONLY);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t w = 0; w < S.n; ++w) {
    if (!is_wall(S, w)) continue;
    double sW = 0, sp = 0, sWr = 0, sr[3] = {0, 0, 0}, sv[3] = {0, 0, 0};
    for (int64_t q = S.nb_off[w]; q < S.nb_off[w + 1]; ++q) {
      int64_t f = S.nb[q];
      if (is_wall(S, f)) continue;
      double d[3], r2 = 0;
      for (int k = 0; k < 3; ++k) {
        d[k] = S.r[3 * w + k] - S.r[3 * f + k];  // r_wf
        r2 += d[k] * d[k];
      }
      double W = kernel_w(dim, h, std::sqrt(r2));
      sW += W;
      if (multi) {
        sp += S.p[f] / S.rho[f] * W;
        sWr += W / S.rho[f];
        for (int k = 0; k < 3; ++k) sr[k] += d[k] * W;
      } else {
        sp += S.p[f] * W;
        for (int k = 0; k < 3; ++k) sr[k] += S.rho[f] * d[k] * W;
      }
      for (int k = 0; k < 3; ++k) sv[k] += S.v[3 * f + k] * W;
    }
    if (sW == 0.0) {
      S.pw[w] = 0.0;
      if (with_velocity)
        for (int k = 0; k < 3; ++k) S.vw[3 * w + k] = vwall[k];   // reading A7
      continue;
    }
    double lever = g[0] * sr[0] + g[1] * sr[1] + g[2] * sr[2];  // (g - a_w) . sum
    S.pw[w] = (sp + lever) / (multi ? sWr : sW);
    if (with_velocity)
      for (int k = 0; k < 3; ++k)
        S.vw[3 * w + k] =
            (S.P.flags & ORC_FLAG_WALL_VEL_MIRROR) ? 2.0 * vwall[k] - sv[k] / sW : vwall[k];
  }
}

// Right state of the pair (i, j): fluid j as is, wall j from (p_w, v_w) with the
// density of reading A5: rho_w(i) = rho0_i + p_w / c_i^2.
struct Right {
  double rho, p, c, V;
  double v[3];
};

inline Right right_state(const Ctx& S, int64_t i, int64_t j) {
  Right R;
  if (is_wall(S, j)) {
    int ph = S.tag[i];
    R.c = S.P.c0[ph];
    R.p = S.pw[j];
    R.rho = S.P.rho0[ph] + S.pw[j] / (R.c * R.c);
    R.V = S.V0;
    for (int k = 0; k < 3; ++k) R.v[k] = S.vw[3 * j + k];
  } else {
    R.c = S.P.c0[S.tag[j]];
    R.p = S.p[j];
    R.rho = S.rho[j];
    R.V = S.m[j] / S.rho[j];
    for (int k = 0; k < 3; ++k) R.v[k] = S.v[3 * j + k];
  }
  return R;
}

// O-5.  PAPER.md:67-95, Eq. 2.7-2.9, vector form with v*.
void pass_continuity(Ctx& S) {
  const int dim = S.P.dim;
  const double h = S.P.h;
  const double w0 = kernel_w(dim, h, 0.0);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < S.n; ++i) {
    if (is_wall(S, i)) continue;
    double sig = w0, acc = 0.0;
    const double ci = S.P.c0[S.tag[i]];
    for (int64_t q = S.nb_off[i]; q < S.nb_off[i + 1]; ++q) {
      int64_t j = S.nb[q];
      double d[3], r2 = 0;
      for (int k = 0; k < 3; ++k) {
        d[k] = S.r[3 * i + k] - S.r[3 * j + k];  // r_ij
        r2 += d[k] * d[k];
      }
      double r = std::sqrt(r2);
      if (counts_in_sigma(S, i, j)) sig += kernel_w(dim, h, r);
      if (r == 0.0) continue;  // reading A21
      Right R = right_state(S, i, j);
      double e[3], UL = 0, UR = 0;
      for (int k = 0; k < 3; ++k) {
        e[k] = -d[k] / r;  // e_ij
        UL += S.v[3 * i + k] * e[k];
        UR += R.v[k] * e[k];
      }
      Riemann s = riemann(S.rho[i], UL, S.p[i], ci, R.rho, UR, R.p, R.c);
      double dw = kernel_dw(dim, h, r);
      double dot = 0;
      for (int k = 0; k < 3; ++k) {
        double vbar = s.wL * S.v[3 * i + k] + s.wR * R.v[k];
        double vstar = s.Ustar * e[k] + (vbar - s.Ubar * e[k]);
        double gradW = dw * d[k] / r;
        dot += (S.v[3 * i + k] - vstar) * gradW;
      }
      acc += 2.0 * S.rho[i] * R.V * dot;  // Eq. 2.9
    }
    S.sigma[i] = sig;
    S.drho[i] = acc;
  }
}

// O-6.  PAPER.md:167-171, Eq. 2.21 (continuity phases), Eq. 2.4 in the normalised
// form of Eq. 2.18 (summation phases, reading A15), then Eq. 2.3.
void density_update(Ctx& S, double dt) {
  for (int64_t i = 0; i < S.n; ++i) {
    if (is_wall(S, i)) continue;
    int ph = S.tag[i];
    if ((S.P.free_surface_mask >> ph) & 1u)
      S.rho[i] += dt * S.drho[i];
    else if (S.P.variant & ORC_VAR_SUM_RAW)
      S.rho[i] = S.m[i] * S.sigma[i];                         // Eq. 2.4 as printed
    else
      S.rho[i] = S.P.rho0[ph] * S.sigma[i] / S.sigma0;        // reading A15
    S.p[i] = S.P.c0[ph] * S.P.c0[ph] * (S.rho[i] - S.P.rho0[ph]);
  }
}

// O-7 (pair part).  PAPER.md:93 Eq. 2.10, :105 Eq. 2.11, :122-137 Eq. 2.13-2.15
// (readings A8, A9, A11, A20).
void pass_momentum(Ctx& S, const double g[3]) {
  const int dim = S.P.dim;
  const double h = S.P.h, dp = S.P.dp;
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < S.n; ++i) {
    if (is_wall(S, i)) {
      S.a[3 * i] = S.a[3 * i + 1] = S.a[3 * i + 2] = 0.0;
      continue;
    }
    const int ph = S.tag[i];
    const double ci = S.P.c0[ph];
    const bool pen = ((S.P.penalty_phase_mask >> ph) & 1u) && !(S.P.flags & ORC_FLAG_WALL_ADAMI_ONLY);
    double a[3] = {g[0], g[1], g[2]};
    if (dim == 2) a[2] = 0.0;
    for (int64_t q = S.nb_off[i]; q < S.nb_off[i + 1]; ++q) {
      int64_t j = S.nb[q];
      double d[3], r2 = 0;
      for (int k = 0; k < 3; ++k) {
        d[k] = S.r[3 * i + k] - S.r[3 * j + k];
        r2 += d[k] * d[k];
      }
      double r = std::sqrt(r2);
      if (r == 0.0) continue;
      double dw = kernel_dw(dim, h, r);
      Right R = right_state(S, i, j);
      double pstar;
      if (is_wall(S, j)) {
        pstar = (S.rho[i] * R.p + R.rho * S.p[i]) / (S.rho[i] + R.rho);  // Eq. 2.11
      } else {
        double UL = 0, UR = 0;
        for (int k = 0; k < 3; ++k) {
          double e = -d[k] / r;
          UL += S.v[3 * i + k] * e;
          UR += R.v[k] * e;
        }
        pstar = riemann(S.rho[i], UL, S.p[i], ci, R.rho, UR, R.p, R.c).pstar;
      }
      for (int k = 0; k < 3; ++k)
        a[k] -= 2.0 * R.V * (pstar / S.rho[i]) * dw * d[k] / r;  // Eq. 2.10
      if (pen && is_wall(S, j)) {
        const double* n = &S.nw[3 * j];
        if (n[0] != 0.0 || n[1] != 0.0 || n[2] != 0.0) {
          double nd = n[0] * d[0] + n[1] * d[1] + n[2] * d[2];  // n_w . (r_i - r_w)
          double sdir = nd / r;
          double delta = 2.0 * nd / dp;
          if (delta < 1.0 && delta > -1.0) {  // reading A9b: only wall particles facing i
            double lam = (1.0 - delta) * (1.0 - delta);
            double Pn = S.P.penalty_strength * lam * std::fabs(S.p[i] * sdir);
            for (int k = 0; k < 3; ++k) a[k] -= 2.0 * (S.V0 / S.rho[i]) * Pn * n[k] * dw;
          }
        }
      }
    }
    for (int k = 0; k < 3; ++k) S.a[3 * i + k] = a[k];
  }
}

void step_once(Ctx& S, double dt) {
  reinitialise(S);                                   // O-1
  for (int64_t i = 0; i < S.n; ++i) {                // O-3, Eq. 2.19-2.20
    if (is_wall(S, i)) continue;
    for (int k = 0; k < S.P.dim; ++k) {
      S.v[3 * i + k] += 0.5 * dt * S.a[3 * i + k];
      S.r[3 * i + k] += dt * S.v[3 * i + k];
    }
  }
  if (walls_move(S)) {                               // NEXT-1: walls at t^{n+1}
    double sdis[3], vwall[3], aw[3];
    wall_motion(S, S.t + dt, sdis, vwall, aw);
    for (int64_t i = 0; i < S.n; ++i)
      if (is_wall(S, i))
        for (int k = 0; k < S.P.dim; ++k) S.r[3 * i + k] = S.r0[3 * i + k] + sdis[k];
  }
  build_neighbours(S);
  double g[3];
  gravity_at(S, S.t + dt, g);                        // reading A28
  wall_extrapolate(S, g, true, S.t + dt);            // O-4
  pass_continuity(S);                                // O-5
  density_update(S, dt);                             // O-6
  wall_extrapolate(S, g, false, S.t + dt);           // O-7 (wall pressure only)
  pass_momentum(S, g);                               // O-7
  for (int64_t i = 0; i < S.n; ++i) {                // O-8, Eq. 2.22
    if (is_wall(S, i)) continue;
    for (int k = 0; k < S.P.dim; ++k) S.v[3 * i + k] += 0.5 * dt * S.a[3 * i + k];
  }
  S.t += dt;
  S.dt_last = dt;
  S.steps++;
}

// --- float32 integer contract (reading A24/A25) ---
struct GridF32 {
  float o[3], inv;
  int nc[3];
  float rc2;
};

GridF32 grid_f32(const orc_params& P) {
  GridF32 G;
  double edge = 2.0 * P.h * (1.0 + 1.0 / 1024.0);
  G.inv = (float)(1.0 / edge);
  for (int k = 0; k < 3; ++k) {
    G.o[k] = (float)P.domain_min[k];
    G.nc[k] = (k < P.dim) ? std::max(1, (int)std::ceil((P.domain_max[k] - P.domain_min[k]) / edge))
                          : 1;
  }
  G.rc2 = (float)(4.0 * P.h * P.h);
  return G;
}

inline int cell_coord_f32(float x, float o, float inv, int n) {
  float u = (x - o);   // one FP32 subtract (compiled with -ffp-contract=off)
  u = u * inv;         // one FP32 multiply
  int c = (int)floorf(u);
  return std::min(std::max(c, 0), n - 1);
}

inline int32_t cell_id_f32(const GridF32& G, int dim, const float* x) {
  int cx = cell_coord_f32(x[0], G.o[0], G.inv, G.nc[0]);
  int cy = cell_coord_f32(x[1], G.o[1], G.inv, G.nc[1]);
  int cz = dim == 3 ? cell_coord_f32(x[2], G.o[2], G.inv, G.nc[2]) : 0;
  return (int32_t)(((int64_t)cz * G.nc[1] + cy) * G.nc[0] + cx);
}

inline float dist2_f32(int dim, const float* a, const float* b) {
  float dx = a[0] - b[0], dy = a[1] - b[1];
  float r2 = fmaf(dy, dy, dx * dx);
  if (dim == 3) {
    float dz = a[2] - b[2];
    r2 = fmaf(dz, dz, r2);
  }
  return r2;
}

}  // namespace

// ===========================================================================
extern "C" {

double orc_kernel_w(int dim, double h, double r) { return kernel_w(dim, h, r); }
double orc_kernel_dw(int dim, double h, double r) { return kernel_dw(dim, h, r); }
double orc_sigma0(int dim, double h, double dp) { return sigma0_lattice(dim, h, dp); }
double orc_reinit_density(double rho_star, double rho0, double sigma, double sigma0, int fs) {
  return reinit_density(rho_star, rho0, sigma, sigma0, fs);
}
// out = {Ustar, pstar, Ubar, wL, wR}; mode 0 = dispatch, 1 = paper Eq. 2.8 (uses cL),
// 2 = acoustic extension.
void orc_riemann(int mode, double rL, double UL, double pL, double cL, double rR, double UR,
                 double pR, double cR, double* out) {
  Riemann s = mode == 1   ? riemann_paper(rL, UL, pL, rR, UR, pR, cL)
              : mode == 2 ? riemann_acoustic(rL, UL, pL, cL, rR, UR, pR, cR)
                          : riemann(rL, UL, pL, cL, rR, UR, pR, cR);
  out[0] = s.Ustar; out[1] = s.pstar; out[2] = s.Ubar; out[3] = s.wL; out[4] = s.wR;
}

void* orc_create(const orc_params* p) {
  Ctx* S = new Ctx();
  S->P = *p;
  S->V0 = std::pow(p->dp, p->dim);
  S->sigma0 = sigma0_lattice(p->dim, p->h, p->dp);
  return S;
}
void orc_destroy(void* h) { delete (Ctx*)h; }

// O-0.  Inputs are float32 (the same arrays the CUDA library receives).
// pos, vel: n*3 (z ignored in 2-D), rho: n, tag: n (phase id, or -1 for wall).
int orc_set_particles(void* hd, int64_t n, const float* pos, const float* vel, const float* rho,
                      const int32_t* tag) {
  Ctx& S = *(Ctx*)hd;
  S.n = n;
  S.r.resize(3 * n); S.v.resize(3 * n); S.a.assign(3 * n, 0.0);
  S.rho.resize(n); S.p.resize(n); S.m.resize(n); S.sigma.resize(n); S.drho.assign(n, 0.0);
  S.tag.assign(tag, tag + n);
  S.pw.assign(n, 0.0); S.vw.assign(3 * n, 0.0); S.nw.assign(3 * n, 0.0);
  for (int64_t i = 0; i < n; ++i) {
    for (int k = 0; k < 3; ++k) {
      bool live = k < S.P.dim;
      S.r[3 * i + k] = live ? (double)pos[3 * i + k] : 0.0;
      S.v[3 * i + k] = (live && tag[i] != ORC_TAG_WALL) ? (double)vel[3 * i + k] : 0.0;
    }
    if (tag[i] == ORC_TAG_WALL) {
      S.rho[i] = S.P.rho0[0]; S.p[i] = 0.0; S.m[i] = S.P.rho0[0] * S.V0;
    } else {
      if (tag[i] < 0 || tag[i] >= S.P.n_phases) return -1;
      int ph = tag[i];
      S.rho[i] = (double)rho[i];
      S.m[i] = S.P.rho0[ph] * S.V0;                                   // reading A19
      S.p[i] = S.P.c0[ph] * S.P.c0[ph] * (S.rho[i] - S.P.rho0[ph]);   // Eq. 2.3
    }
  }
  S.r0 = S.r;
  S.t = S.P.t_start; S.steps = 0; S.dt_last = 0;
  build_neighbours(S);
  wall_normals(S);
  number_density(S);
  double g[3];
  gravity_at(S, S.t, g);
  wall_extrapolate(S, g, true, S.t);
  pass_momentum(S, g);   // (dv/dt)^0, reading A18
  return 0;
}

// dt_in == NULL: Eq. 2.23-2.24 each step.  dt_out (optional) receives the dt used.
int orc_step(void* hd, int32_t nsteps, const double* dt_in, double* dt_out) {
  Ctx& S = *(Ctx*)hd;
  for (int s = 0; s < nsteps; ++s) {
    double dt = dt_in ? dt_in[s] : time_step(S);
    if (dt_out) dt_out[s] = dt;
    step_once(S, dt);
  }
  return 0;
}

// Any pointer may be NULL.  Original particle order.  Wall entries: vel = v_w,
// rho = rho0[0] + p_w/c0[0]^2, p = p_w, acc = 0.
void orc_get_fields(void* hd, double* pos, double* vel, double* rho, double* p, double* acc,
                    double* sigma, double* drho) {
  Ctx& S = *(Ctx*)hd;
  for (int64_t i = 0; i < S.n; ++i) {
    bool w = is_wall(S, i);
    for (int k = 0; k < 3; ++k) {
      if (pos) pos[3 * i + k] = S.r[3 * i + k];
      if (vel) vel[3 * i + k] = w ? S.vw[3 * i + k] : S.v[3 * i + k];
      if (acc) acc[3 * i + k] = S.a[3 * i + k];
    }
    if (rho) rho[i] = w ? S.P.rho0[0] + S.pw[i] / (S.P.c0[0] * S.P.c0[0]) : S.rho[i];
    if (p) p[i] = w ? S.pw[i] : S.p[i];
    if (sigma) sigma[i] = S.sigma[i];
    if (drho) drho[i] = S.drho[i];
  }
}

void orc_get_normals(void* hd, double* nw) {
  Ctx& S = *(Ctx*)hd;
  std::copy(S.nw.begin(), S.nw.end(), nw);
}

// out[8] = {t, dt_last, steps, npairs, E_k, mass, x_front, escaped}
// x_front = max x over phase-0 particles within 3 dp of the lowest live axis origin
// (floor = domain_min[dim-1] + 3 dp wall band).
void orc_get_stats(void* hd, double* out) {
  Ctx& S = *(Ctx*)hd;
  double ek = 0, mass = 0, xf = -1e300;
  int up = S.P.dim - 1;
  double floor_z = S.P.domain_min[up] + 3.0 * S.P.dp;
  for (int64_t i = 0; i < S.n; ++i) {
    if (is_wall(S, i)) continue;
    double v2 = 0;
    for (int k = 0; k < 3; ++k) v2 += S.v[3 * i + k] * S.v[3 * i + k];
    ek += 0.5 * S.m[i] * v2;
    mass += S.m[i];
    if (S.tag[i] == 0 && S.r[3 * i + up] < floor_z + 3.0 * S.P.dp)
      xf = std::max(xf, S.r[3 * i]);
  }
  out[0] = S.t; out[1] = S.dt_last; out[2] = (double)S.steps; out[3] = (double)S.npairs;
  out[4] = ek; out[5] = mass; out[6] = xf; out[7] = (double)S.escaped;
}

int64_t orc_neighbour_count(void* hd) { return (int64_t)((Ctx*)hd)->nb.size(); }
void orc_get_neighbours(void* hd, int64_t* off, int32_t* ids) {
  Ctx& S = *(Ctx*)hd;
  std::copy(S.nb_off.begin(), S.nb_off.end(), off);
  std::copy(S.nb.begin(), S.nb.end(), ids);
}

// Brute-force all-pairs neighbour count/list in double on the current positions (pin P6).
// ids may be NULL (count only).  Returns the total.
int64_t orc_neighbours_bruteforce(void* hd, int64_t* off, int32_t* ids) {
  Ctx& S = *(Ctx*)hd;
  double rc2 = 4.0 * S.P.h * S.P.h;
  int64_t tot = 0;
  for (int64_t i = 0; i < S.n; ++i) {
    off[i] = tot;
    for (int64_t j = 0; j < S.n; ++j) {
      if (j == i) continue;
      double d2 = 0;
      for (int k = 0; k < 3; ++k) {
        double d = S.r[3 * i + k] - S.r[3 * j + k];
        d2 += d * d;
      }
      if (d2 < rc2) {
        if (ids) ids[tot] = (int32_t)j;
        tot++;
      }
    }
  }
  off[S.n] = tot;
  return tot;
}

// ---- float32 integer contract: cell ids, permutation, cell ranges, lists ----
// Layout: fluid and wall particles are indexed on
// the same grid but sorted separately.  cell_id[n] in caller order; perm[n] =
// [fluid ids stably sorted by cell | wall ids stably sorted by cell];
// cell_start/cell_end [2*ncell]: fluid grid then wall grid, positions relative to
// the start of the class's block in perm.
int64_t orc_f32_ncell(const orc_params* P) {
  GridF32 G = grid_f32(*P);
  return (int64_t)G.nc[0] * G.nc[1] * G.nc[2];
}

void orc_f32_cells(const orc_params* P, int64_t n, const float* pos, const int32_t* tag,
                   int32_t* cell_id, int32_t* perm, int32_t* cell_start, int32_t* cell_end) {
  GridF32 G = grid_f32(*P);
  int64_t ncell = (int64_t)G.nc[0] * G.nc[1] * G.nc[2];
  for (int64_t i = 0; i < n; ++i) cell_id[i] = cell_id_f32(G, P->dim, &pos[3 * i]);
  int64_t base = 0;
  for (int cls = 0; cls < 2; ++cls) {
    std::vector<int32_t> ids;
    for (int64_t i = 0; i < n; ++i)
      if ((tag[i] == ORC_TAG_WALL) == (cls == 1)) ids.push_back((int32_t)i);
    std::stable_sort(ids.begin(), ids.end(),
                     [&](int32_t a, int32_t b) { return cell_id[a] < cell_id[b]; });
    int32_t* cs = cell_start + cls * ncell;
    int32_t* ce = cell_end + cls * ncell;
    for (int64_t c = 0; c < ncell; ++c) cs[c] = ce[c] = 0;
    for (size_t s = 0; s < ids.size(); ++s) {
      perm[base + s] = ids[s];
      int32_t c = cell_id[ids[s]];
      if (s == 0 || cell_id[ids[s - 1]] != c) cs[c] = (int32_t)s;
      ce[c] = (int32_t)s + 1;
    }
    base += (int64_t)ids.size();
  }
}

// Neighbour lists by the FP32 rule r2 = fmaf(dz,dz,fmaf(dy,dy,dx*dx)) < (float)(4h^2):
// fluid i: all j != i of any tag; wall i: fluid j only.  Ids ascending.  Brute force.
int64_t orc_f32_neighbours(const orc_params* P, int64_t n, const float* pos, const int32_t* tag,
                           int64_t* off, int32_t* ids, int64_t cap) {
  GridF32 G = grid_f32(*P);
  int64_t tot = 0;
  for (int64_t i = 0; i < n; ++i) {
    off[i] = tot;
    bool wi = tag[i] == ORC_TAG_WALL;
    for (int64_t j = 0; j < n; ++j) {
      if (j == i) continue;
      if (wi && tag[j] == ORC_TAG_WALL) continue;
      if (dist2_f32(P->dim, &pos[3 * i], &pos[3 * j]) < G.rc2) {
        if (ids && tot < cap) ids[tot] = (int32_t)j;
        tot++;
      }
    }
  }
  off[n] = tot;
  return tot;
}

// Same lists through the float32 cell grid (27 / 9 cell walk); used to check that the
// grid never loses a pair that the brute-force rule finds.
int64_t orc_f32_neighbours_grid(const orc_params* P, int64_t n, const float* pos,
                                const int32_t* tag, int64_t* off, int32_t* ids, int64_t cap) {
  GridF32 G = grid_f32(*P);
  int64_t ncell = (int64_t)G.nc[0] * G.nc[1] * G.nc[2];
  std::vector<int32_t> cid(n);
  std::vector<int64_t> start(ncell + 1, 0);
  for (int64_t i = 0; i < n; ++i) {
    cid[i] = cell_id_f32(G, P->dim, &pos[3 * i]);
    start[cid[i] + 1]++;
  }
  for (int64_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
  std::vector<int32_t> order(n);
  {
    std::vector<int64_t> fill(start.begin(), start.end() - 1);
    for (int64_t i = 0; i < n; ++i) order[fill[cid[i]]++] = (int32_t)i;
  }
  int64_t tot = 0;
  std::vector<int32_t> li;
  for (int64_t i = 0; i < n; ++i) {
    off[i] = tot;
    li.clear();
    bool wi = tag[i] == ORC_TAG_WALL;
    int c = cid[i];
    int cx = c % G.nc[0], cy = (c / G.nc[0]) % G.nc[1], cz = c / (G.nc[0] * G.nc[1]);
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          int x = cx + dx, y = cy + dy, z = cz + dz;
          if (x < 0 || y < 0 || z < 0 || x >= G.nc[0] || y >= G.nc[1] || z >= G.nc[2]) continue;
          int64_t cc = ((int64_t)z * G.nc[1] + y) * G.nc[0] + x;
          for (int64_t s = start[cc]; s < start[cc + 1]; ++s) {
            int32_t j = order[s];
            if (j == i) continue;
            if (wi && tag[j] == ORC_TAG_WALL) continue;
            if (dist2_f32(P->dim, &pos[3 * i], &pos[3 * j]) < G.rc2) li.push_back(j);
          }
        }
    std::sort(li.begin(), li.end());
    for (int32_t j : li) {
      if (ids && tot < cap) ids[tot] = j;
      tot++;
    }
  }
  off[n] = tot;
  return tot;
}

}  // extern "C"
