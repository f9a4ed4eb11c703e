/*
 * tslb.h -- C ABI of the B200-native thread-safe lattice Boltzmann (TSLB) two-component time
 * step of arxiv 2403.15773 ("PAPER.md" below = /root/reference/PAPER.md; readings A1..A18 are
 * listed in DESIGN.md §3).
 *
 * One context owns the state of one simulation on one CUDA device:
 *   per lattice node   rho, u = (ux,uy,uz), Pi^neq = (xx,yy,zz,xy,xz,yz)   [PAPER.md:108]
 *   and, if two_component, the phase field phi                              [PAPER.md:198-211]
 * double-buffered in device memory (HBM).  No populations f_i are ever stored.  tslb_step()
 * advances all nodes by n time steps; per step every node pulls its 26 neighbours' stored moments,
 * rebuilds their post-collision D3Q27 populations f^eq + (1-omega) f^neq with the third-order
 * Hermite expansion (eq. 5, 98 eq. 6, 166 eq. 16, 183 eq. 19), takes the moments of
 * the streamed populations, and advances phi by the D3Q7 LB of PAPER.md:206-211
 * eqs. 23-24 with the surface-tension force F = sigma kappa grad(phi) (PAPER.md:192-196
 * eqs. 20-21) applied as a velocity kick.  Every step runs in hand-written CUDA kernels for
 * sm_100a; there is no CPU fallback.
 *
 * Conventions
 *   - Every function returns TSLB_OK (0) or a negative error code; nothing throws or aborts.
 *     tslb_last_error() returns a human-readable description of the last failure.
 *   - Field arrays passed in/out are DENSE, x fastest: element (x,y,z) at x + nx*(y + ny*z),
 *     nx*ny*nz elements of the context's precision (float for TSLB_F32, double for TSLB_F64).
 *   - Pointers are HOST pointers when pointers_on_device == 0 and DEVICE pointers (same device
 *     as the context) when it is 1.  The caller owns every buffer it passes; the library copies
 *     in / out and keeps no caller pointer except `workspace` and `stream`.
 *   - All device work is enqueued on `stream`.  tslb_step() is asynchronous; tslb_get_moments()
 *     synchronises the stream before returning.
 *   - x and y are always periodic.  z is periodic, or jet inflow at z = 0 with outflow at
 *     z = nz-1 (eqs. 9-10, 223); a z face can also be shared with another
 *     context that holds the neighbouring z-slab (TSLB_BC_HALO, "z-slabs" below).
 */
#ifndef TSLB_H
#define TSLB_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tslb_ctx tslb_ctx; /* opaque, owned by the library */

enum { TSLB_OK = 0, TSLB_EINVAL = -1, TSLB_ENOMEM = -2, TSLB_ECUDA = -3, TSLB_ESTATE = -4 };
enum { TSLB_F32 = 0, TSLB_F64 = 1 };
/* z face types.  TSLB_BC_HALO marks a face shared with a neighbouring z-slab of a multi-GPU run
 * (see "z-slabs" below): the context then keeps two ghost planes behind that face, which the
 * neighbour fills.  Allowed pairs (zlo, zhi): PERIODIC/PERIODIC, JET_INFLOW/OUTFLOW, and with
 * slabs HALO/HALO, JET_INFLOW/HALO, HALO/OUTFLOW.                                                */
enum { TSLB_BC_PERIODIC = 0, TSLB_BC_JET_INFLOW = 1, TSLB_BC_OUTFLOW = 2, TSLB_BC_HALO = 3 };
/* kernel selection (tslb_params.kernel) */
enum {
  TSLB_KERNEL_AUTO = 0,     /* fastest kernel that supports the grid                           */
  TSLB_KERNEL_GENERIC = 1,  /* one thread per node, direct global loads; any grid size         */
  TSLB_KERNEL_TILED = 2     /* TMA-staged 32x8 x-y tiles (two-component fp64: 32x6) marching along z;
                               needs nx >= 32, ny >= 8 (two-component fp64: 6) and nx a multiple of 4
                               (fp32) / 2 (fp64), field arrays at most 8 GB apart; a ragged last tile is
                               shifted back inside the grid (tslb_create fails with TSLB_EINVAL
                               when the grid is not supported)                                 */
};

/* How the surface-tension force F = sigma kappa grad(phi) (eq. 20) enters the flow
 * solver.  The paper does not say; both readings are listed in DESIGN.md §3.
 *   TSLB_FORCING_KICK (A9, default): after streaming, u' = u_b + F/rho' with F from the OLD phi;
 *     the collision is built on u'.  Stored velocity: u'.  All kernels.
 *   TSLB_FORCING_GUO (A18): time-centred forcing of Guo, Zheng & Shi, Phys. Rev. E
 *     65 (2002) 046308.  At every source node the collision is built on u = u_b + F/(2 rho) with
 *     the F of the same time level and carries the source populations (1 - omega/2) S_i,
 *     S_i = w_i [(c_i - u).F/c_s^2 + (c_i.u)(c_i.F)/c_s^4]; phi is advected with u.  Stored
 *     velocity: the bare u_b = m/rho (so tslb_init_fields takes u_b and tslb_get_moments returns
 *     it).  F on a source node needs phi three nodes away, beyond the 2-node phi halo of the tiled
 *     kernel: this reading runs on TSLB_KERNEL_GENERIC only (F in three scratch arrays), needs
 *     two_component, and does not take TSLB_BC_HALO faces.                                      */
enum { TSLB_FORCING_KICK = 0, TSLB_FORCING_GUO = 1 };

typedef struct {
  int nx, ny, nz;          /* grid.  All > 0; nz >= 4 if z is not periodic */
  int precision;           /* TSLB_F32 | TSLB_F64: element type of every field pointer and
                              the arithmetic type of the kernels                               */
  int two_component;       /* 0: flow only; 1: flow + phase field           */
  int hermite_order;       /* 3: eqs. 16 and 19 (the paper's scheme); 2: eq. 8                 */
  double omega;            /* relaxation frequency, 0 < omega < 2;
                              nu = c_s^2 (1/omega - 1/2), c_s^2 = 1/3            */
  double sigma;            /* surface tension of eq. 20                         */
  double interface_width;  /* W > 0: equilibrium profile phi = 1/2 (1 + tanh(2 s / W));
                              anti-diffusion gamma of eq. 24 is 2/W (reading A8)               */
  int bc_zlo, bc_zhi;      /* TSLB_BC_PERIODIC / TSLB_BC_PERIODIC, or
                              TSLB_BC_JET_INFLOW / TSLB_BC_OUTFLOW                             */
  double jet_diameter;     /* D: nozzle disc (x-(nx-1)/2)^2 + (y-(ny-1)/2)^2 < (D/2)^2 on z=0  */
  double jet_velocity;     /* U: inflow u_z = U (1 + jet_perturbation * xi)                    */
  double jet_perturbation; /* amplitude of the seeded uniform perturbation xi in (-1,1) (A12)  */
  unsigned long long seed; /* seed of the counter-based inflow hash                            */
  int device;              /* CUDA device ordinal                                              */
  int kernel;              /* TSLB_KERNEL_*                                                    */
  void *stream;            /* cudaStream_t of the caller (NULL = legacy default stream)        */
  void *workspace;         /* optional caller-owned DEVICE memory, 256-byte aligned (e.g. a
                              torch tensor); NULL -> the library allocates with cudaMalloc     */
  size_t workspace_bytes;  /* size of `workspace`; must be >= tslb_workspace_bytes()           */
  int forcing;             /* TSLB_FORCING_KICK | TSLB_FORCING_GUO                             */
} tslb_params;

/* Device bytes the context needs: 2 buffers (the paper's rule "read the fields of time t, write elsewhere",
 * PAPER.md:94-96, 213, kept as double buffering) x (10 moment arrays rho, u, Pi^neq -- what the method
 * stores per node, PAPER.md:108 -- [+ phi, PAPER.md:198-211]) in the padded internal layout (x/y ghost
 * cells for the periodic wrap), plus scratch arrays of the generic kernel.  Host
 * function, no device work.  0 if the parameters are invalid.                                       */
size_t tslb_workspace_bytes(const tslb_params *p);

/* Create a context for the problem the paper states: grid, relaxation frequency
 * omega <-> nu = c_s^2 (1/omega - 1/2), surface tension sigma (eq. 20),
 * interface width, boundary types (eqs. 9-10, 223).  Validates the
 * parameters (TSLB_EINVAL: sizes <= 0, omega outside (0,2), sigma < 0 or not finite, W <= 0 when
 * two_component, |jet_velocity| >= 1, jet_perturbation outside [0,1], nz < 4 with inflow/outflow,
 * unsupported face pair, kernel/forcing combination), selects the device (TSLB_ECUDA when there is no
 * sm_100 device: no CPU fallback), allocates the workspace with cudaMalloc or adopts the caller's
 * (TSLB_ENOMEM / TSLB_EINVAL), builds the TMA descriptors of the tiled kernel.  On failure *out is NULL
 * and tslb_last_error(NULL) returns the message of the failed create (per thread).  The context keeps
 * `workspace` and `stream`; both must outlive it.                                                    */
int tslb_create(const tslb_params *p, tslb_ctx **out);

/* Set the time-0 state and reset the step counter.  The state IS the collision-ready moments of
 * the first collision builds f^eq(rho, u) + (1 - omega) f^neq(Pi^neq, u) from them
 * (eq. 5), so Pi^neq = 0 is a plain equilibrium start.  rho, ux, uy, uz: required.  phi:
 * required iff two_component (else must be NULL; TSLB_EINVAL).  pineq: NULL (-> Pi^neq = 0) or 6
 * pointers xx,yy,zz,xy,xz,yz (NULL entries -> 0).  With inflow/outflow the two z boundary planes are
 * then set from the initial fields as in a step (eqs. 9-10, readings A10/A11; hash
 * step index 0).  Copies the caller's arrays (host arrays through a pinned-free staging buffer);
 * synchronises the stream.                                                                           */
int tslb_init_fields(tslb_ctx *c, const void *rho, const void *ux, const void *uy, const void *uz,
                     const void *phi, const void *const pineq[6], int pointers_on_device);

/* Advance nsteps >= 0 time steps (eq. 6 + 206 eq. 23 per step).  Asynchronous on
 * the context's stream.  TSLB_ESTATE before tslb_init_fields.  From nsteps = 5 on (and on a stream
 * other than the legacy default stream) the steps are replayed from a CUDA graph of two steps that the
 * context captures once per starting buffer, so that small grids are not bound by kernel launches;
 * the first such call allocates an 8-byte device counter.  Do not call it with nsteps >= 5 while the
 * stream is itself being captured.                                                                  */
int tslb_step(tslb_ctx *c, int nsteps);

/* Copy out the stored state -- the moments the method keeps per node and phi
 * (PAPER.md:198-211): rho, the stored velocity (KICK: the post-kick u'; GUO: the bare u_b;
 * see tslb_get_physical_velocity), Pi^neq (NOT the full Pi; reading A2; relative to u_b) and phi.  Any
 * pointer (and any entry of pineq, or pineq itself) may be NULL.  Synchronises the stream.      */
int tslb_get_moments(tslb_ctx *c, void *rho, void *ux, void *uy, void *uz, void *const pineq[6],
                     void *phi, int pointers_on_device);

/* The time-centred ("physical") velocity of the current state, (m_pre + m_post)/(2 rho): the mean of
 * the momentum before and after the forced collision.  KICK: u' - F/(2 rho) with the F that made
 * the last kick (from phi of the previous step, still held in the other buffer; F = 0 before the
 * first step); GUO: u_b + F/(2 rho) with F of the current phi.  F = 0 on inflow/outflow planes and
 * when !two_component.  Runs the phase-geometry kernels of the generic path into three scratch
 * arrays (allocated on first use for a tiled context).  Any pointer may be NULL.  Synchronises the
 * stream.  Not available on a z-slab (TSLB_EINVAL).                                              */
int tslb_get_physical_velocity(tslb_ctx *c, void *ux, void *uy, void *uz, int pointers_on_device);

/* The same velocity for callers that must not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): this entry point calls no cudaMalloc, cudaFree or allocating
 * library routine.  ux, uy, uz are DEVICE pointers (dense, nx*ny*nz elements of the context's precision;
 * any may be NULL); the call is asynchronous on the context's stream and does NOT synchronise it.  The
 * scratch it needs (the three normal arrays n = grad(phi)/(|grad(phi)|+eps), eqs. 20-21,
 * of the padded grid) is one file-scope device array of tslb_noalloc_scratch_bytes() = 12 MiB that every
 * GPU holds from the moment it loads the library until the process exits; its device address is resolved
 * once per device (cudaGetSymbolAddress) when a context is created there.  Grids that need more --
 * 3 * (nx+16)*(ny+4)*nz elements, each array rounded up to 256 bytes -- are rejected with TSLB_EINVAL and
 * a message (about 1.0 M padded nodes in fp32, 0.5 M in fp64: e.g. 64x64x128 fp32, 64^3 fp64).  All
 * contexts on a device SHARE the array and it keeps the last call's contents (every entry a call reads
 * it has written first, so nothing is cleared): two calls that overlap on the GPU -- different streams,
 * or different contexts on one device -- race; serialise them.  TSLB_EINVAL on a z-slab.             */
int tslb_get_physical_velocity_noalloc(tslb_ctx *c, void *ux, void *uy, void *uz);
size_t tslb_noalloc_scratch_bytes(void);

/* ---- z-slabs: one domain split along z over several contexts / GPUs (the paper's
 * stated next step).  Every node update reads only time-t values within one
 * plane (moments) / two planes (phi) of itself, so a slab needs, per step and per shared face, the
 * neighbour's face plane of the 10 moments and its two planes of phi.  There is no exchange
 * kernel and no pack/unpack: the step kernel of a slab stores those planes, besides its own
 * time-t+1 buffer, straight into the neighbour's ghost planes through peer pointers (same process:
 * the neighbour's workspace pointer; other process: a CUDA IPC handle of it; other GPU: NVLink
 * peer stores).  Protocol (all slabs in lockstep):
 *     create each slab with TSLB_BC_HALO on its shared faces, the same nx, ny, precision,
 *     two_component and kernel; attach the neighbours; tslb_init_fields on every slab;
 *     [barrier]  tslb_halo_push on every slab  [barrier]
 *     repeat:  tslb_step(c, 1) on every slab;  [barrier: all slabs finished step t]
 * The barrier must order the streams (same stream, an event, a tiny NCCL all-reduce on the
 * stream, or a host barrier after a stream synchronise); tslb_step refuses nsteps > 1 on a slab.
 * The inflow hash is keyed by (x, y, step) only, so a slab run reproduces the single-context run
 * bit for bit.                                                                                    */

/* Base device pointer of the context's workspace (to hand to a neighbour in the same process).  */
void *tslb_workspace_ptr(const tslb_ctx *c);

/* Declare the slab behind `face` (0: z low, 1: z high), whose workspace starts at device pointer
 * nb_workspace (valid on this context's device: same device, peer-mapped, or IPC-opened) and
 * which has nb_nz planes.  TSLB_EINVAL if the face is not a TSLB_BC_HALO face.  The pointer is
 * kept until tslb_destroy; the neighbour must outlive this context's last step.                 */
int tslb_attach_neighbor(tslb_ctx *c, int face, void *nb_workspace, int nb_nz);

/* The same across processes: export this context's workspace as a 64-byte CUDA IPC handle (host
 * buffer; needs a library-allocated workspace) / attach a neighbour from such a handle.         */
int tslb_ipc_get_handle(tslb_ctx *c, void *handle64);
int tslb_attach_neighbor_ipc(tslb_ctx *c, int face, const void *handle64, int nb_nz);

/* Forget the attached neighbours (synchronises the stream; closes handles opened by
 * tslb_attach_neighbor_ipc).  Tear-down across processes is two-phase: every rank detaches, a
 * barrier, then every rank destroys -- CUDA forbids freeing exported memory that an importer still
 * has open.  tslb_step on a detached halo face fails with TSLB_ESTATE.                             */
int tslb_detach_neighbors(tslb_ctx *c);

/* Copy the face planes of the CURRENT buffer into the attached neighbours' ghost planes
 * (asynchronous on the stream).  Needed once after tslb_init_fields; afterwards tslb_step keeps
 * the ghost planes current by itself.                                                           */
int tslb_halo_push(tslb_ctx *c);

/* ---- time averages on the mid x-z plane (Figs. 5-6: the time-averaged phase
 * field and axial velocity, from which the centre-line 1/<phi_c>, 1/<u_c> and the radial profiles
 * follow).  After tslb_stats_begin(c, every), every `every`-th time step adds phi and u_z of the
 * plane y = (ny-1)/2 (the mean of the two middle rows when ny is even: the jet axis lies between
 * them) to fp64 running sums, by a small kernel on the context's stream.  tslb_stats_get copies
 * the sums (HOST pointers, nx*nz doubles each, element (x,z) at x + nx*z; either may be NULL;
 * sum_phi is left untouched when !two_component) and the number of samples; <q> = sum / nsamples.
 * tslb_stats_begin again restarts the sums; tslb_stats_end stops accumulating.  A z-slab
 * accumulates its own planes.                                                                    */
int tslb_stats_begin(tslb_ctx *c, int every);
int tslb_stats_get(tslb_ctx *c, double *sum_phi, double *sum_uz, long long *nsamples);
int tslb_stats_end(tslb_ctx *c);

/* Number of time steps taken since tslb_init_fields (keys the inflow hash).                     */
long long tslb_step_count(const tslb_ctx *c);

/* Name of the kernel tslb_step launches for this context ("generic", "tiled<64x8>", ...) and the
 * number of kernel launches it has made so far (for benchmark bookkeeping).                     */
const char *tslb_kernel_name(const tslb_ctx *c);
long long tslb_launch_count(const tslb_ctx *c);

/* Inflow perturbation xi(seed, x, y, step) in (-1,1) evaluated ON THE DEVICE for x in [0,nx),
 * y in [0,ny) into out[nx*ny] doubles (host pointer) -- test probe for the bit-exact hash pin.  */
int tslb_debug_xi(tslb_ctx *c, long long step, double *out_host);

/* Test probe for the arithmetic of 1/rho' and |grad(phi)| in the tiled kernel ("fp32 / fp64
 * arithmetic of 1/rho' and n"): evaluates, ON THE DEVICE and in the context's precision, the kernel's reciprocal and
 * square root of in[0..n) (host doubles, converted to the context's precision) into out_rcp[n] and out_sqrt[n] (host
 * doubles).  Synchronous; allocates and frees its own scratch.  TSLB_EINVAL for a NULL argument or n < 1.             */
int tslb_debug_math(tslb_ctx *c, int n, const double *in_host, double *out_rcp_host, double *out_sqrt_host);

/* Synchronise the stream, close imported neighbour handles, free what the library allocated (not a
 * caller-owned workspace).  NULL is accepted.  Always TSLB_OK.                                      */
int tslb_destroy(tslb_ctx *c);

/* Last error message of the context (or of the last failed tslb_create when c == NULL).
 * The string is owned by the library and valid until the next call on the same context/thread.  */
const char *tslb_last_error(const tslb_ctx *c);

#ifdef __cplusplus
}
#endif
#endif /* TSLB_H */
