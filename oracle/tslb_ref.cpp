/*
 * tslb_ref.cpp -- plain, slow, fp64 CPU ORACLE of the two-component TSLB step.
 *
 * TEST INFRASTRUCTURE ONLY (see tslb_ref.h).  No code shared with the CUDA path.
 *
 * What it is: the paper's algorithm written out literally.  Full D3Q27 populations are stored
 * (27 per node), streamed (eq. 1), their moments taken, and the
 * post-collision state rebuilt as f^eq + (1-omega) f^neq (eq. 5, 98 eq. 6) with the
 * third-order Hermite equilibrium (eq. 16) and the third-order regularized
 * non-equilibrium (eq. 19, read as in DESIGN.md A3/A4), both evaluated by explicit
 * sums over the tensor indices alpha,beta,gamma -- no closed forms, no symmetry tricks, no tiling.
 * The phase field is the D3Q7 LB of PAPER.md:206-211 eqs. 23-24 (only its zeroth moment is needed
 * because the relaxation time is one), and the surface-tension force is eq. 20-21 in CSF form
 * (A6/A7/A9).  Boundary nodes follow PAPER.md:125-137 eqs. 9-10 (A10/A11).
 *
 * Numerical note N1: populations are kept in deviation form f_i - w_i and the density as
 * drho = rho - 1.  This is the same arithmetic (everything is linear in the rest state) and keeps
 * Pi^neq from being formed as a small difference of O(1/3) numbers.
 *
 * A second forcing reading (A18, Guo-type time-centred forcing; tslb_ref.h TSLB_REF_FORCING_GUO) is
 * implemented beside the kick of A9: collide_guo() / step_once() branches marked GUO.  The paper
 * is silent on how the force enters; A18 is pinned by the published scheme's moment conditions,
 * momentum balance, closed-form forced flows and a numpy restatement (tests/test_oracle_forcing.py).
 *
 * Parity pins: tests/test_oracle_*.py (one named pin per function: DESIGN.md section 2).  The inflow /
 * outflow READING (A10, A11: which values are imposed on the two planes, and from which time level) is
 * not fixed by the paper; what boundary_planes() does with that reading is pinned: the populations it
 * rebuilds are eq. 9 (test_jet_boundary_populations_are_eq9), the interior mass changes by exactly what
 * they carry in and out and the inlet flux is sum_nozzle rho_B U (1 + p xi)
 * (test_jet_mass_balance_from_boundary_populations), and under A18 the two planes carry no force
 * (test_guo_jet_momentum_balance_with_unforced_boundary_planes).
 */
#include "tslb_ref.h"

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double CS2 = 1.0 / 3.0;          /* c_s^2 */
const double CS2G = 1.0 / 4.0;         /* D3Q7 c_{s,g}^2, reading A8 */
const double EPS_N = 1e-12;            /* regulariser of |grad phi|, reading A7 */

struct Lattice {
  int c[27][3];
  double w[27];
  double H2[27][3][3];                 /* c c - c_s^2 delta            (eq. 7)  */
  double H3[27][3][3][3];              /* third Hermite tensor         (eq. 16) */
  int c7[7][3];
  double w7[7];
  Lattice() {
    const double w1[3] = {1.0 / 6.0, 2.0 / 3.0, 1.0 / 6.0}; /* 1-D weights of -1, 0, +1 (A1) */
    for (int k = 0; k < 3; ++k)
      for (int j = 0; j < 3; ++j)
        for (int i = 0; i < 3; ++i) {
          int q = i + 3 * j + 9 * k;
          c[q][0] = i - 1; c[q][1] = j - 1; c[q][2] = k - 1;
          w[q] = w1[i] * w1[j] * w1[k];
        }
    for (int q = 0; q < 27; ++q)
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
          double dab = (a == b) ? 1.0 : 0.0;
          H2[q][a][b] = c[q][a] * c[q][b] - CS2 * dab;
          for (int g = 0; g < 3; ++g) {
            double dbg = (b == g) ? 1.0 : 0.0, dag = (a == g) ? 1.0 : 0.0;
            H3[q][a][b][g] = (double)(c[q][a] * c[q][b] * c[q][g]) -
                             CS2 * (c[q][g] * dab + c[q][a] * dbg + c[q][b] * dag);
          }
        }
    /* D3Q7: rest + six face vectors, w0 = 1/4, w = 1/8 (A8) */
    const int f[7][3] = {{0, 0, 0}, {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1}};
    for (int q = 0; q < 7; ++q) {
      for (int a = 0; a < 3; ++a) c7[q][a] = f[q][a];
      w7[q] = (q == 0) ? 0.25 : 0.125;
    }
  }
};
const Lattice L;

/* f_i^eq - w_i, eq. 16 by explicit tensor sums (order 2: eq. 2). */
void feq_dev(double drho, const double u[3], int order, double out[27]) {
  const double rho = 1.0 + drho;
  for (int q = 0; q < 27; ++q) {
    double t1 = 0.0, t2 = 0.0, t3 = 0.0;
    for (int a = 0; a < 3; ++a) t1 += L.c[q][a] * u[a];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) t2 += L.H2[q][a][b] * u[a] * u[b];
    if (order >= 3)
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
          for (int g = 0; g < 3; ++g) t3 += L.H3[q][a][b][g] * u[a] * u[b] * u[g];
    out[q] = L.w[q] * (drho + rho * (t1 / CS2 + t2 / (2.0 * CS2 * CS2) + t3 / (6.0 * CS2 * CS2 * CS2)));
  }
}

/* f_i^neq, eq. 19 with the Hermite form of eqs. 7/12 (A3): w_i prefactor and
 * H^2 = c c - c_s^2 delta; a^3 is the symmetric three-term recursion of eq. 19 (A4). */
void fneq(const double a2[3][3], const double u[3], int order, double out[27]) {
  for (int q = 0; q < 27; ++q) {
    double t2 = 0.0, t3 = 0.0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) t2 += L.H2[q][a][b] * a2[a][b];
    if (order >= 3)
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
          for (int g = 0; g < 3; ++g) {
            double a3 = a2[a][b] * u[g] + u[a] * a2[b][g] + u[b] * a2[a][g];
            t3 += L.H3[q][a][b][g] * a3;
          }
    out[q] = L.w[q] * (t2 / (2.0 * CS2 * CS2) + t3 / (6.0 * CS2 * CS2 * CS2));
  }
}

void sym6_to_33(const double p[6], double a[3][3]) { /* xx,yy,zz,xy,xz,yz */
  a[0][0] = p[0]; a[1][1] = p[1]; a[2][2] = p[2];
  a[0][1] = a[1][0] = p[3]; a[0][2] = a[2][0] = p[4]; a[1][2] = a[2][1] = p[5];
}

/* Counter-based inflow perturbation (A12): splitmix64 finaliser of seed + (counter+1)*golden,
 * top 24 bits k -> xi = (2k + 1 - 2^24) / 2^24 in (-1, 1). */
double xi_hash(uint64_t seed, int x, int y, int nx, int ny, int64_t step) {
  uint64_t counter = (uint64_t)step * ((uint64_t)nx * (uint64_t)ny) + (uint64_t)(x + nx * y);
  uint64_t z = seed + (counter + 1ULL) * 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  z = z ^ (z >> 31);
  int64_t k = (int64_t)(z >> 40);
  int64_t num = 2 * k + 1 - (1LL << 24);
  return (double)num / 16777216.0;
}

}  // namespace

struct tslb_ref_ctx {
  tslb_ref_params p;
  size_t N;
  bool zper;
  double gamma;
  int64_t t;
  bool inited;
  std::vector<double> fpost, fpost2;        /* 27*N, deviation form f - w        */
  std::vector<double> rho, u, pineq, phi;   /* N, 3N, 6N, N  (time-t fields)     */
  std::vector<double> rho2, u2, pineq2, phi2;
  std::vector<double> G, nrm, kappa;        /* 3N, 3N, N (phase geometry, old phi) */
  std::vector<double> Fext;                 /* 3N or empty: pin-only extra force density      */
  std::vector<double> Ftot;                 /* 3N: KICK: force of the last kick; GUO: force of
                                               the current fields (the one in fpost)          */
  std::vector<double> drho_s;               /* N (GUO): rho - 1 exactly as the moment sum gave it */
  bool guo;

  inline int wrapx(int x) const { return (x % p.nx + p.nx) % p.nx; }
  inline int wrapy(int y) const { return (y % p.ny + p.ny) % p.ny; }
  inline int mapz(int z) const { /* periodic wrap, or clamp (O5/O8) */
    if (zper) return (z % p.nz + p.nz) % p.nz;
    return z < 0 ? 0 : (z >= p.nz ? p.nz - 1 : z);
  }
  inline size_t idx(int x, int y, int z) const {
    return (size_t)x + (size_t)p.nx * ((size_t)y + (size_t)p.ny * (size_t)z);
  }
  inline bool is_boundary(int z) const { return !zper && (z == 0 || z == p.nz - 1); }

  /* O5: G = (1/c_s^2) sum_i w_i c_i phi(x+c_i), n = G/(|G|+eps) for all nodes; then
   * kappa = -(1/c_s^2) sum_i w_i c_i . n(x+c_i)   (eqs. 20-21, A6/A7). */
  void phase_geometry() {
    const int nx = p.nx, ny = p.ny, nz = p.nz;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          double g[3] = {0, 0, 0};
          for (int q = 0; q < 27; ++q) {
            size_t j = idx(wrapx(x + L.c[q][0]), wrapy(y + L.c[q][1]), mapz(z + L.c[q][2]));
            for (int a = 0; a < 3; ++a) g[a] += L.w[q] * L.c[q][a] * phi[j];
          }
          for (int a = 0; a < 3; ++a) g[a] /= CS2;
          double mag = std::sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
          size_t i = idx(x, y, z);
          for (int a = 0; a < 3; ++a) {
            G[a * N + i] = g[a];
            nrm[a * N + i] = g[a] / (mag + EPS_N);
          }
        }
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          double d = 0.0;
          for (int q = 0; q < 27; ++q) {
            size_t j = idx(wrapx(x + L.c[q][0]), wrapy(y + L.c[q][1]), mapz(z + L.c[q][2]));
            for (int a = 0; a < 3; ++a) d += L.w[q] * L.c[q][a] * nrm[a * N + j];
          }
          kappa[idx(x, y, z)] = -d / CS2;
        }
  }

  /* O2+O3+O7: post-collision populations of one node from its collision-ready moments. */
  void collide_node(size_t i, double drho, const double uu[3], const double pn[6], double *dst) const {
    double fe[27], fn[27], a2[3][3];
    sym6_to_33(pn, a2);
    feq_dev(drho, uu, p.hermite_order, fe);
    fneq(a2, uu, p.hermite_order, fn);
    for (int q = 0; q < 27; ++q) dst[(size_t)q * N + i] = fe[q] + (1.0 - p.omega) * fn[q];
  }

  /* Force density of the CURRENT fields: F = sigma kappa G (eq. 20, A6/A7) from the
   * current phi [+ the pin-only extra force]; zero on inflow/outflow planes (their moments are
   * imposed, O9).  Also leaves n of the current phi in nrm. */
  void compute_force() {
    const bool two = p.two_component != 0;
    if (two) phase_geometry();
    for (int a = 0; a < 3; ++a)
      for (size_t i = 0; i < N; ++i) {
        double F = two ? p.sigma * kappa[i] * G[a * N + i] : 0.0;
        if (!Fext.empty()) F += Fext[a * N + i];
        Ftot[a * N + i] = F;
      }
    if (!zper)
      for (int a = 0; a < 3; ++a)
        for (int y = 0; y < p.ny; ++y)
          for (int x = 0; x < p.nx; ++x)
            Ftot[a * N + idx(x, y, 0)] = Ftot[a * N + idx(x, y, p.nz - 1)] = 0.0;
  }

  /* Reading A18: collision with the forcing of Guo, Zheng & Shi (2002).  From the
   * bare moments rho, u_b = m/rho, Pi_b^neq = Pi - rho c_s^2 delta - rho u_b u_b of the streamed
   * populations and the force F of the same time level:
   *   u      = u_b + F / (2 rho)                                  (Guo eq. 19: rho u = m + F/2)
   *   Pi^neq = Pi - rho c_s^2 delta - rho u u                     (second moment of f - f^eq(u);
   *            Guo's (uF + Fu)/2 belongs to the viscous-stress diagnostic, not to the relaxation)
   *   f^pre  = f^eq(rho,u) + f^neq(Pi^neq,u) + w_i c_i.(m - rho u)/c_s^2,   m - rho u = -F/2
   *            (regularized pre-collision state, eqs. 16/19 + the first-order Hermite term that
   *            carries the momentum defect of f^eq(u))
   *   f^post = f^eq + (1-omega)(f^pre - f^eq) + (1 - omega/2) S_i                (Guo eq. 4, 20)
   *   S_i    = w_i [ (c_i - u).F / c_s^2 + (c_i.u)(c_i.F) / c_s^4 ]
   * With F = 0 this is collide_node bit for bit. */
  void collide_guo(size_t i, double drho, const double ub[3], const double pn[6], const double F[3],
                   double *dst) const {
    const double rho = 1.0 + drho;
    double uu[3], a2b[3][3], a2[3][3], fe[27], fn[27];
    for (int a = 0; a < 3; ++a) uu[a] = ub[a] + F[a] / (2.0 * rho);
    sym6_to_33(pn, a2b);
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        a2[a][b] = a2b[a][b] + (rho * ub[a] * ub[b] - rho * uu[a] * uu[b]);
    feq_dev(drho, uu, p.hermite_order, fe);
    fneq(a2, uu, p.hermite_order, fn);
    double uF = 0.0;
    for (int a = 0; a < 3; ++a) uF += uu[a] * F[a];
    for (int q = 0; q < 27; ++q) {
      double cF = 0.0, cu = 0.0;
      for (int a = 0; a < 3; ++a) { cF += L.c[q][a] * F[a]; cu += L.c[q][a] * uu[a]; }
      const double first = L.w[q] * (-0.5 * cF) / CS2;
      const double S = L.w[q] * ((cF - uF) / CS2 + cu * cF / (CS2 * CS2));
      dst[(size_t)q * N + i] = fe[q] + (1.0 - p.omega) * (fn[q] + first) + (1.0 - 0.5 * p.omega) * S;
    }
  }

  void collide_all_guo() {
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)N; ++i) {
      const double ub[3] = {u[i], u[N + i], u[2 * N + i]};
      const double F[3] = {Ftot[i], Ftot[N + i], Ftot[2 * N + i]};
      double pn[6];
      for (int k = 0; k < 6; ++k) pn[k] = pineq[k * N + i];
      collide_guo((size_t)i, drho_s[i], ub, pn, F, fpost.data());
    }
  }

  /* O9: moments imposed on the two z boundary planes, from time-t ("old") fields in r,uo,po,ph
   * (eqs. 9-10; A10, A11).  step_index keys the inflow hash. */
  void boundary_planes(const std::vector<double> &r, const std::vector<double> &uo,
                       const std::vector<double> &po, const std::vector<double> &ph,
                       std::vector<double> &rn, std::vector<double> &un, std::vector<double> &pn,
                       std::vector<double> &phn, std::vector<double> &fdst, int64_t step_index) {
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const double D = p.jet_diameter;
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        /* inflow plane z = 0: u imposed, rho and Pi^neq from the fluid neighbour z = 1 */
        {
          size_t b = idx(x, y, 0), f = idx(x, y, 1);
          long long ix = 2LL * x - (nx - 1), iy = 2LL * y - (ny - 1); /* 2*(x - centre) */
          bool inside = (double)(ix * ix + iy * iy) < D * D;         /* r^2 < (D/2)^2   */
          double uu[3] = {0.0, 0.0, 0.0};
          if (inside)
            uu[2] = p.jet_velocity * (1.0 + p.jet_perturbation * xi_hash(p.seed, x, y, nx, ny, step_index));
          double pi6[6];
          for (int k = 0; k < 6; ++k) pi6[k] = po[k * N + f];
          rn[b] = r[f];
          for (int a = 0; a < 3; ++a) un[a * N + b] = uu[a];
          for (int k = 0; k < 6; ++k) pn[k * N + b] = pi6[k];
          if (p.two_component) phn[b] = inside ? 1.0 : 0.0;
          collide_node(b, rn[b] - 1.0, uu, pi6, fdst.data());
        }
        /* outflow plane z = nz-1: rho = 1, the rest copied from z = nz-2 */
        {
          size_t b = idx(x, y, nz - 1), f = idx(x, y, nz - 2);
          double uu[3], pi6[6];
          for (int a = 0; a < 3; ++a) uu[a] = uo[a * N + f];
          for (int k = 0; k < 6; ++k) pi6[k] = po[k * N + f];
          rn[b] = 1.0;
          for (int a = 0; a < 3; ++a) un[a * N + b] = uu[a];
          for (int k = 0; k < 6; ++k) pn[k * N + b] = pi6[k];
          if (p.two_component) phn[b] = ph[f];
          collide_node(b, 0.0, uu, pi6, fdst.data());
        }
      }
  }

  void step_once() {
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const bool two = p.two_component != 0;
    const bool forced = two || !Fext.empty();
    /* KICK: O5, force and n from the OLD phi.  GUO: Ftot and nrm already belong to the current
     * (time-t) fields -- they were formed for the collision that produced fpost. */
    if (!guo) compute_force();
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z) {
      if (is_boundary(z)) continue; /* overwritten in O9; their pulled values are never used */
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          const size_t i = idx(x, y, z);
          /* O1 stream (pull): f_i(x) = fpost_i(x - c_i)      PAPER.md:71 eq. 1, 98 eq. 6 */
          double f[27];
          for (int q = 0; q < 27; ++q) {
            size_t j = idx(wrapx(x - L.c[q][0]), wrapy(y - L.c[q][1]), mapz(z - L.c[q][2]));
            f[q] = fpost[(size_t)q * N + j];
          }
          /* O4 bare moments */
          double drho = 0.0, m[3] = {0, 0, 0}, P[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
          for (int q = 0; q < 27; ++q) {
            drho += f[q];
            for (int a = 0; a < 3; ++a) {
              m[a] += L.c[q][a] * f[q];
              for (int b = 0; b < 3; ++b) P[a][b] += L.c[q][a] * L.c[q][b] * f[q];
            }
          }
          const double rh = 1.0 + drho;
          double ub[3];
          for (int a = 0; a < 3; ++a) ub[a] = m[a] / rh;
          /* Pi^neq' = Pi' - rho' u_b u_b - rho' c_s^2 delta; in deviation form P holds
           * Pi' - c_s^2 delta, so the O(1/3) term cancels analytically (N1). */
          double a2[3][3];
          for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b)
              a2[a][b] = P[a][b] - rh * ub[a] * ub[b] - ((a == b) ? drho * CS2 : 0.0);
          /* O5/O6 force and kick                              PAPER.md:192 eq. 20; A9 */
          double un[3] = {ub[0], ub[1], ub[2]};
          if (forced && !guo)
            for (int a = 0; a < 3; ++a) un[a] += Ftot[a * N + i] / rh;
          /* O2+O3+O7 collide                                  PAPER.md:91 eq. 5
           * (GUO: the bare moments are stored; the collision follows once F(t+1) is known) */
          const double pn[6] = {a2[0][0], a2[1][1], a2[2][2], a2[0][1], a2[0][2], a2[1][2]};
          if (!guo) collide_node(i, drho, un, pn, fpost2.data());
          else drho_s[i] = drho;
          rho2[i] = rh;
          for (int a = 0; a < 3; ++a) u2[a * N + i] = un[a];
          for (int k = 0; k < 6; ++k) pineq2[k * N + i] = pn[k];
          /* O8 phase step: OLD phi, OLD stored u, n from OLD phi   PAPER.md:206-211 eqs. 23-24 */
          if (two) {
            double s = 0.0;
            for (int q = 0; q < 7; ++q) {
              size_t j = idx(wrapx(x - L.c7[q][0]), wrapy(y - L.c7[q][1]), mapz(z - L.c7[q][2]));
              double cu = 0.0, cn = 0.0;
              for (int a = 0; a < 3; ++a) {
                /* advecting velocity: the stored one (KICK, A9) / the time-centred physical
                 * velocity u_b + F/(2 rho) of the source node (GUO, A18) */
                double ua = u[a * N + j];
                if (guo) ua += Ftot[a * N + j] / (2.0 * rho[j]);
                cu += L.c7[q][a] * ua;
                cn += L.c7[q][a] * nrm[a * N + j];
              }
              double ph = phi[j];
              s += L.w7[q] * ph * (1.0 + cu / CS2G) + L.w7[q] * gamma * ph * (1.0 - ph) * cn;
            }
            phi2[i] = s;
          }
        }
    }
    if (!zper) boundary_planes(rho, u, pineq, phi, rho2, u2, pineq2, phi2, fpost2, t + 1);
    if (!guo) fpost.swap(fpost2);
    rho.swap(rho2); u.swap(u2); pineq.swap(pineq2);
    if (two) phi.swap(phi2);
    ++t;
    if (guo) {
      if (!zper)
        for (int y = 0; y < ny; ++y)
          for (int x = 0; x < nx; ++x) {
            drho_s[idx(x, y, 0)] = rho[idx(x, y, 0)] - 1.0;
            drho_s[idx(x, y, nz - 1)] = rho[idx(x, y, nz - 1)] - 1.0;
          }
      compute_force();     /* F(t+1), n(t+1) from the new phi */
      collide_all_guo();   /* fpost(t+1), boundary planes included (F = 0 there) */
    }
  }
};

extern "C" {

int tslb_ref_create(const tslb_ref_params *p, tslb_ref_ctx **out) {
  if (!p || !out) return -1;
  *out = nullptr;
  if (p->nx <= 0 || p->ny <= 0 || p->nz <= 0) return -1;
  if (!(p->omega > 0.0 && p->omega < 2.0)) return -1;
  if (p->hermite_order != 2 && p->hermite_order != 3) return -1;
  if (p->two_component && !(p->interface_width > 0.0)) return -1;
  bool zper = (p->bc_zlo == TSLB_REF_BC_PERIODIC && p->bc_zhi == TSLB_REF_BC_PERIODIC);
  bool jet = (p->bc_zlo == TSLB_REF_BC_JET_INFLOW && p->bc_zhi == TSLB_REF_BC_OUTFLOW);
  if (!zper && !jet) return -1;
  if (jet && p->nz < 4) return -1;
  if (p->forcing != TSLB_REF_FORCING_KICK && p->forcing != TSLB_REF_FORCING_GUO) return -1;
  tslb_ref_ctx *c = new (std::nothrow) tslb_ref_ctx();
  if (!c) return -2;
  c->p = *p;
  c->N = (size_t)p->nx * p->ny * p->nz;
  c->zper = zper;
  c->gamma = p->two_component ? 2.0 / p->interface_width : 0.0;
  c->t = 0;
  c->inited = false;
  c->guo = p->forcing == TSLB_REF_FORCING_GUO;
  try {
    const size_t N = c->N;
    c->fpost.assign(27 * N, 0.0); c->fpost2.assign(27 * N, 0.0);
    c->rho.assign(N, 1.0); c->rho2.assign(N, 1.0);
    c->u.assign(3 * N, 0.0); c->u2.assign(3 * N, 0.0);
    c->pineq.assign(6 * N, 0.0); c->pineq2.assign(6 * N, 0.0);
    c->Ftot.assign(3 * N, 0.0);
    c->drho_s.assign(N, 0.0);
    if (p->two_component) {
      c->phi.assign(N, 0.0); c->phi2.assign(N, 0.0);
      c->G.assign(3 * N, 0.0); c->nrm.assign(3 * N, 0.0); c->kappa.assign(N, 0.0);
    }
  } catch (...) {
    delete c;
    return -2;
  }
  *out = c;
  return 0;
}

int tslb_ref_init_fields(tslb_ref_ctx *c, const double *rho, const double *ux, const double *uy,
                         const double *uz, const double *phi, const double *const pineq[6]) {
  if (!c || !rho || !ux || !uy || !uz) return -1;
  if (c->p.two_component && !phi) return -1;
  const size_t N = c->N;
  std::memcpy(c->rho.data(), rho, N * sizeof(double));
  std::memcpy(c->u.data(), ux, N * sizeof(double));
  std::memcpy(c->u.data() + N, uy, N * sizeof(double));
  std::memcpy(c->u.data() + 2 * N, uz, N * sizeof(double));
  for (int k = 0; k < 6; ++k) {
    if (pineq && pineq[k]) std::memcpy(c->pineq.data() + k * N, pineq[k], N * sizeof(double));
    else std::fill(c->pineq.begin() + k * N, c->pineq.begin() + (k + 1) * N, 0.0);
  }
  if (c->p.two_component) std::memcpy(c->phi.data(), phi, N * sizeof(double));
  /* fpost = f^eq(rho0,u0) + (1-omega) f^neq(Pi^neq0,u0) */
#pragma omp parallel for schedule(static)
  for (long long i = 0; i < (long long)N; ++i) {
    double uu[3] = {c->u[i], c->u[N + i], c->u[2 * N + i]};
    double pn[6];
    for (int k = 0; k < 6; ++k) pn[k] = c->pineq[k * N + i];
    c->collide_node((size_t)i, c->rho[i] - 1.0, uu, pn, c->fpost.data());
  }
  c->t = 0;
  if (!c->zper) {
    /* boundary planes from the initial fields themselves, hash step index 0 */
    std::vector<double> r0 = c->rho, u0 = c->u, p0 = c->pineq, ph0 = c->phi;
    c->boundary_planes(r0, u0, p0, ph0, c->rho, c->u, c->pineq, c->phi, c->fpost, 0);
  }
  std::fill(c->Ftot.begin(), c->Ftot.end(), 0.0);
  if (c->guo) {
    /* the given velocity is the stored (bare) one; F(0) from phi(0) enters the first collision */
    for (size_t i = 0; i < N; ++i) c->drho_s[i] = c->rho[i] - 1.0;
    c->compute_force();
    c->collide_all_guo();
  }
  c->inited = true;
  return 0;
}

int tslb_ref_step(tslb_ref_ctx *c, int nsteps) {
  if (!c || nsteps < 0) return -1;
  if (!c->inited) return -4;
  for (int s = 0; s < nsteps; ++s) c->step_once();
  return 0;
}

int tslb_ref_get_moments(tslb_ref_ctx *c, double *rho, double *ux, double *uy, double *uz,
                         double *const pineq[6], double *phi) {
  if (!c) return -1;
  if (!c->inited) return -4;
  const size_t N = c->N;
  if (rho) std::memcpy(rho, c->rho.data(), N * sizeof(double));
  if (ux) std::memcpy(ux, c->u.data(), N * sizeof(double));
  if (uy) std::memcpy(uy, c->u.data() + N, N * sizeof(double));
  if (uz) std::memcpy(uz, c->u.data() + 2 * N, N * sizeof(double));
  if (pineq)
    for (int k = 0; k < 6; ++k)
      if (pineq[k]) std::memcpy(pineq[k], c->pineq.data() + k * N, N * sizeof(double));
  if (phi) {
    if (!c->p.two_component) return -1;
    std::memcpy(phi, c->phi.data(), N * sizeof(double));
  }
  return 0;
}

int tslb_ref_destroy(tslb_ref_ctx *c) {
  delete c;
  return 0;
}

void tslb_ref_lattice(int *cc, double *w) {
  for (int q = 0; q < 27; ++q) {
    for (int a = 0; a < 3; ++a) cc[3 * q + a] = L.c[q][a];
    w[q] = L.w[q];
  }
}

void tslb_ref_feq(double rho, const double u[3], int order, double out[27]) {
  feq_dev(rho - 1.0, u, order, out);
  for (int q = 0; q < 27; ++q) out[q] += L.w[q];
}

void tslb_ref_fneq(const double pineq[6], const double u[3], int order, double out[27]) {
  double a2[3][3];
  sym6_to_33(pineq, a2);
  fneq(a2, u, order, out);
}

int tslb_ref_get_populations(tslb_ref_ctx *c, double *fpost) {
  if (!c || !fpost) return -1;
  for (int q = 0; q < 27; ++q)
    for (size_t i = 0; i < c->N; ++i) fpost[(size_t)q * c->N + i] = c->fpost[(size_t)q * c->N + i] + L.w[q];
  return 0;
}

int tslb_ref_phase_geometry(tslb_ref_ctx *c, double *G, double *n, double *kappa, double *F) {
  if (!c || !c->p.two_component) return -1;
  c->phase_geometry();
  const size_t N = c->N;
  if (G) std::memcpy(G, c->G.data(), 3 * N * sizeof(double));
  if (n) std::memcpy(n, c->nrm.data(), 3 * N * sizeof(double));
  if (kappa) std::memcpy(kappa, c->kappa.data(), N * sizeof(double));
  if (F)
    for (int a = 0; a < 3; ++a)
      for (size_t i = 0; i < N; ++i) F[a * N + i] = c->p.sigma * c->kappa[i] * c->G[a * N + i];
  return 0;
}

int tslb_ref_set_extra_force(tslb_ref_ctx *c, const double *Fext) {
  if (!c) return -1;
  if (!Fext) { c->Fext.clear(); return 0; }
  c->Fext.assign(Fext, Fext + 3 * c->N);
  return 0;
}

int tslb_ref_get_physical_velocity(tslb_ref_ctx *c, double *ux, double *uy, double *uz) {
  if (!c) return -1;
  if (!c->inited) return -4;
  const size_t N = c->N;
  double *out[3] = {ux, uy, uz};
  const double sgn = c->guo ? 0.5 : -0.5;
  for (int a = 0; a < 3; ++a)
    if (out[a])
      for (size_t i = 0; i < N; ++i) out[a][i] = c->u[a * N + i] + sgn * c->Ftot[a * N + i] / c->rho[i];
  return 0;
}

double tslb_ref_xi(unsigned long long seed, int x, int y, int nx, int ny, long long step) {
  return xi_hash((uint64_t)seed, x, y, nx, ny, (int64_t)step);
}

int tslb_ref_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
