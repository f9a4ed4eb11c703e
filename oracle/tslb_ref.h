/*
 * tslb_ref.h -- C ABI of the CPU ORACLE for the two-component thread-safe lattice Boltzmann
 * (TSLB) time step of arxiv 2403.15773.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may load it.  It shares no code, header,
 * table or constant with the CUDA path under paper_2403_15773_b200/csrc/.
 *
 * Everything is fp64, host memory, dense x-fastest arrays of nx*ny*nz doubles
 * (linear index x + nx*(y + ny*z)).  The oracle stores the full D3Q27 post-collision
 * populations (eq. 1, 98 eq. 6) and applies the third-order regularized collision
 * exactly as PAPER.md:166 eq. 16 and PAPER.md:183 eq. 19 define it (readings: DESIGN.md §3).
 */
#ifndef TSLB_REF_H
#define TSLB_REF_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tslb_ref_ctx tslb_ref_ctx;

enum { TSLB_REF_BC_PERIODIC = 0, TSLB_REF_BC_JET_INFLOW = 1, TSLB_REF_BC_OUTFLOW = 2 };
/* How the force F = sigma kappa grad(phi) (eq. 20) enters the flow solver.  The paper
 * does not say; both readings are listed in DESIGN.md §3.
 *   KICK (A9, the default): velocity kick u' = u_b + F/rho' after streaming, F from the OLD phi.
 *   GUO  (A18): time-centred forcing of Guo, Zheng & Shi, Phys. Rev. E 65 (2002)
 *        046308: collision velocity u = (m + F/2)/rho, source populations (1 - omega/2) S_i with
 *        S_i = w_i [ (c_i - u).F / c_s^2 + (c_i.u)(c_i.F) / c_s^4 ],  F evaluated at the time level
 *        of the populations being collided.  Stored velocity: the bare u_b = m/rho.              */
enum { TSLB_REF_FORCING_KICK = 0, TSLB_REF_FORCING_GUO = 1 };

typedef struct {
  int nx, ny, nz;          /* grid; x and y always periodic                                 */
  int two_component;       /* 0: flow only; 1: flow + phase field                           */
  int hermite_order;       /* 3 (eqs. 16, 19) or 2 (eq. 8)                                  */
  double omega;            /* relaxation frequency, nu = c_s^2 (1/omega - 1/2) PAPER.md:87  */
  double sigma;            /* surface tension (eq. 20)                                      */
  double interface_width;  /* W; anti-diffusion gamma = 2/W (reading A8)          */
  int bc_zlo, bc_zhi;      /* PERIODIC/PERIODIC or JET_INFLOW/OUTFLOW                       */
  double jet_diameter, jet_velocity, jet_perturbation;
  unsigned long long seed; /* inflow perturbation seed (reading A12)                        */
  int forcing;             /* TSLB_REF_FORCING_KICK | TSLB_REF_FORCING_GUO                  */
} tslb_ref_params;

/* All return 0 on success, negative on error. */
int tslb_ref_create(const tslb_ref_params *p, tslb_ref_ctx **out);
/* phi may be NULL when !two_component; pineq may be NULL (zeros) -- 6 arrays xx,yy,zz,xy,xz,yz */
int tslb_ref_init_fields(tslb_ref_ctx *c, const double *rho, const double *ux, const double *uy,
                         const double *uz, const double *phi, const double *const pineq[6]);
int tslb_ref_step(tslb_ref_ctx *c, int nsteps);
/* any output pointer may be NULL */
int tslb_ref_get_moments(tslb_ref_ctx *c, double *rho, double *ux, double *uy, double *uz,
                         double *const pineq[6], double *phi);
int tslb_ref_destroy(tslb_ref_ctx *c);

/* ---- probes used only by the pin tests ---- */
/* lattice: c[27][3] (as 81 ints, i-major), w[27] */
void tslb_ref_lattice(int *c, double *w);
/* f_i^eq (eq. 16; order 2 -> PAPER.md:76 eq. 2) and f_i^neq (eq. 19 as read in A3) */
void tslb_ref_feq(double rho, const double u[3], int order, double out[27]);
void tslb_ref_fneq(const double pineq[6], const double u[3], int order, double out[27]);
/* full post-collision populations (w_i added back), 27 arrays of N, i-major */
int tslb_ref_get_populations(tslb_ref_ctx *c, double *fpost);
/* phase geometry of the CURRENT phi (eqs. 20-21 as read in A6/A7): G[3N], n[3N], kappa[N], F[3N] */
int tslb_ref_phase_geometry(tslb_ref_ctx *c, double *G, double *n, double *kappa, double *F);
/* Pin-only probe: a static force density Fext (3N doubles, component-major; NULL clears it) that
 * is ADDED to sigma kappa grad(phi) at every interior node (also when !two_component).  The method
 * has no such term; it lets the forcing be pinned on flows with a closed form (uniform
 * acceleration, Kolmogorov flow).  Call before tslb_ref_init_fields. */
int tslb_ref_set_extra_force(tslb_ref_ctx *c, const double *Fext);
/* Time-centred physical velocity of the CURRENT state: KICK: u' - F/(2 rho) with the F that made
 * the last kick (0 before the first step); GUO: u_b + F/(2 rho) with F of the current phi. */
int tslb_ref_get_physical_velocity(tslb_ref_ctx *c, double *ux, double *uy, double *uz);
/* inflow perturbation xi in (-1,1) (reading A12) */
double tslb_ref_xi(unsigned long long seed, int x, int y, int nx, int ny, long long step);
/* number of OpenMP threads the step loop uses */
int tslb_ref_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
