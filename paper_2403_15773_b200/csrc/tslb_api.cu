// tslb_api.cu -- the C-ABI boundary (include/tslb.h): context, validation, workspace carving,
// field import/export, kernel dispatch.  Host-side bookkeeping only; every step of the method
// runs in the kernels of tslb_generic.cuh / tslb_tiled.cuh.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "../../include/tslb.h"
#include "tslb_generic.cuh"
#include "tslb_tiled.cuh"

#include <type_traits>

using namespace tslb;

namespace {

thread_local std::string g_create_error;

size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

Layout make_layout(int nx, int ny, int nz, int gz) {
  Layout L;
  L.nx = nx; L.ny = ny; L.nz = nz;
  L.px = nx + 2 * GX;
  L.py = ny + 2 * GY;
  L.gz = gz;
  L.plane = (long long)L.px * L.py;
  L.field = (long long)round_up((size_t)L.plane * (nz + 2 * gz), 64);
  return L;
}

// Carving of a workspace into the 2 x nfields field arrays; the pointers are those of plane 0 (after
// the gz ghost planes).  The same function locates a NEIGHBOUR slab's arrays from its workspace base.
void carve_fields(void *ws, const Layout &L, size_t esize, int nfields, void *fields[2][NF_MAX], size_t *end) {
  const size_t fb = round_up((size_t)L.field * esize, 256);
  const size_t z0 = (size_t)L.gz * (size_t)L.plane * esize;
  char *base = (char *)ws;
  size_t off = 0;
  for (int b = 0; b < 2; ++b)
    for (int k = 0; k < nfields; ++k) { fields[b][k] = base + off + z0; off += fb; }
  if (end) *end = off;
}

struct Validated {
  bool ok = false;
  std::string why;
  bool zper = true;
  bool slab = false;                  // at least one z face is a halo face
  bool halo_lo = false, halo_hi = false, jet_lo = false, out_hi = false;
  int kernel = TSLB_KERNEL_GENERIC;   // resolved kernel
  size_t esize = 4;
  int nfields = 10;
  Layout L{};
  size_t bytes = 0;
};

Validated validate(const tslb_params *p) {
  Validated v;
  auto fail = [&](const char *m) { v.ok = false; v.why = m; return v; };
  if (!p) return fail("params is NULL");
  if (p->nx <= 0 || p->ny <= 0 || p->nz <= 0) return fail("grid sizes must be positive");
  if ((long long)p->nx * p->ny * p->nz > (1LL << 40)) return fail("grid too large");
  if (p->precision != TSLB_F32 && p->precision != TSLB_F64) return fail("precision must be TSLB_F32 or TSLB_F64");
  if (p->hermite_order != 2 && p->hermite_order != 3) return fail("hermite_order must be 2 or 3");
  if (!(p->omega > 0.0 && p->omega < 2.0)) return fail("omega must be in (0,2)");
  if (p->two_component && !(p->interface_width > 0.0)) return fail("interface_width must be > 0 when two_component");
  const bool zper = p->bc_zlo == TSLB_BC_PERIODIC && p->bc_zhi == TSLB_BC_PERIODIC;
  const bool jet = p->bc_zlo == TSLB_BC_JET_INFLOW && p->bc_zhi == TSLB_BC_OUTFLOW;
  v.halo_lo = p->bc_zlo == TSLB_BC_HALO;
  v.halo_hi = p->bc_zhi == TSLB_BC_HALO;
  v.slab = v.halo_lo || v.halo_hi;
  v.jet_lo = p->bc_zlo == TSLB_BC_JET_INFLOW;
  v.out_hi = p->bc_zhi == TSLB_BC_OUTFLOW;
  if (v.slab) {
    if (!(v.halo_lo || v.jet_lo) || !(v.halo_hi || v.out_hi))
      return fail("a slab face is TSLB_BC_HALO, or JET_INFLOW (z low) / OUTFLOW (z high)");
    if (p->nz < 2) return fail("a slab needs nz >= 2 (the halo is two planes deep)");
    // the imposed plane is not pushed to the neighbour: with nz == 2 it would be the neighbour's second
    // ghost plane of phi, which would go stale
    if ((v.jet_lo || v.out_hi) && p->nz < 3) return fail("a slab with an inflow or outflow face needs nz >= 3");
  } else {
    if (!zper && !jet) return fail("boundary types must be PERIODIC/PERIODIC or JET_INFLOW/OUTFLOW (or TSLB_BC_HALO faces)");
    if (jet && p->nz < 4) return fail("nz >= 4 is required with inflow/outflow");
  }
  if ((v.jet_lo || v.out_hi) && !(p->jet_diameter >= 0.0 && p->jet_diameter < 1e9)) return fail("jet_diameter must be finite and >= 0");
  if (!(p->sigma >= 0.0 && p->sigma < 1e30)) return fail("sigma must be finite and >= 0");
  if (!(p->jet_velocity > -1.0 && p->jet_velocity < 1.0)) return fail("jet_velocity must be finite and |U| < 1 (lattice units)");
  if (!(p->jet_perturbation >= 0.0 && p->jet_perturbation <= 1.0)) return fail("jet_perturbation must be in [0, 1]");
  if (p->two_component && !(p->interface_width < 1e9)) return fail("interface_width must be finite");
  if (p->kernel < TSLB_KERNEL_AUTO || p->kernel > TSLB_KERNEL_TILED) return fail("unknown kernel selector");
  if (p->forcing != TSLB_FORCING_KICK && p->forcing != TSLB_FORCING_GUO) return fail("unknown forcing selector");
  const bool guo = p->forcing == TSLB_FORCING_GUO;
  if (guo && !p->two_component) return fail("TSLB_FORCING_GUO needs two_component (the force comes from phi)");
  if (guo && v.slab) return fail("TSLB_FORCING_GUO does not take TSLB_BC_HALO faces");
  if (guo && p->kernel == TSLB_KERNEL_TILED)
    return fail("TSLB_FORCING_GUO runs on TSLB_KERNEL_GENERIC only (the force on a source node needs a 3-node phi halo)");
  v.zper = zper;
  v.esize = p->precision == TSLB_F32 ? 4 : 8;
  v.nfields = p->two_component ? 11 : 10;
  v.L = make_layout(p->nx, p->ny, p->nz, v.slab ? GZ : 0);
  const bool tiled_ok = tiled_supported(p->precision, p->two_component != 0, p->nx, p->ny, p->nz);
  if (p->kernel == TSLB_KERNEL_TILED && !tiled_ok)
    return fail("TSLB_KERNEL_TILED needs nx >= 32, ny >= 8 (two-component fp64: 6) and nx a multiple of 4 (fp32) or 2 (fp64)");
  v.kernel = (p->kernel == TSLB_KERNEL_GENERIC || !tiled_ok || guo) ? TSLB_KERNEL_GENERIC : TSLB_KERNEL_TILED;
  // 2 buffers x nfields arrays, + 3 scratch arrays (n) for the generic two-component path,
  // + 3 more (F) for TSLB_FORCING_GUO
  size_t narr = 2 * (size_t)v.nfields;
  if (v.kernel == TSLB_KERNEL_GENERIC && p->two_component) narr += 3;
  if (guo) narr += 3;
  v.bytes = narr * round_up((size_t)v.L.field * v.esize, 256);
  v.ok = true;
  return v;
}

}  // namespace

struct tslb_ctx {
  tslb_params p;
  Validated v;
  cudaStream_t stream = nullptr;
  void *ws = nullptr;
  bool own_ws = false;
  void *fields[2][NF_MAX] = {};
  void *nrm[3] = {};
  void *frc[3] = {};           // TSLB_FORCING_GUO: scratch force arrays
  void *nrm_own = nullptr;     // scratch n allocated by tslb_get_physical_velocity on a tiled context
  void *nb_fields[2][2][NF_MAX] = {};   // [side][buffer][field]: neighbour slabs' arrays (peer pointers)
  int nb_nz[2] = {0, 0};
  bool nb_on[2] = {false, false};
  void *nb_ipc[2] = {nullptr, nullptr}; // bases opened with cudaIpcOpenMemHandle
  unsigned char nb_handle[2][64] = {};
  int cur = 0;                 // index of the buffer holding time t
  bool inited = false;
  long long t = 0;
  long long launches = 0;
  void *stage[2] = {nullptr, nullptr};   // two dense fields, for host <-> device import/export: the copy of one
                                          // field overlaps the (un)packing of the other
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
  void *pv_tmp = nullptr;      // tslb_get_physical_velocity to host pointers: three dense fields, kept
  double *stat = nullptr;      // mid-plane running sums: [0] phi, [1] u_z, nx*nz doubles each
  int stat_every = 0;          // 0: off
  long long stat_n = 0;        // samples accumulated
  TiledPlan tiled;             // TMA descriptors etc.
  // tslb_step(n) as a replayed CUDA graph of two steps (buffer 0 -> 1 -> 0 or 1 -> 0 -> 1); the kernels read
  // the step index from step_ctr, which a one-thread kernel advances before every step
  cudaGraphExec_t gexec[2] = {nullptr, nullptr};
  long long *step_ctr = nullptr;
  bool graph_failed = false;
  std::string err;
  std::string kname;

  int fail(int code, const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    err = buf;
    return code;
  }
  int cuda_fail(cudaError_t e, const char *what) {
    return fail(TSLB_ECUDA, "%s: %s", what, cudaGetErrorString(e));
  }
};

#define CK(call)                                             \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return c->cuda_fail(e_, #call);   \
  } while (0)

namespace {

template <typename T>
StepParams<T> make_step_params(tslb_ctx *c, int src, int dst) {
  StepParams<T> P;
  P.L = c->v.L;
  for (int k = 0; k < NF_MAX; ++k) {
    P.in.f[k] = (T *)c->fields[src][k];
    P.out.f[k] = (T *)c->fields[dst][k];
  }
  for (int k = 0; k < 3; ++k) { P.nrm[k] = (T *)c->nrm[k]; P.frc[k] = (T *)c->frc[k]; }
  P.omc = (T)(1.0 - c->p.omega);
  P.sigma = (T)(c->p.two_component ? c->p.sigma : 0.0);
  P.gamma = (T)(c->p.two_component ? 2.0 / c->p.interface_width : 0.0);
  P.zper = c->v.zper ? 1 : 0;
  P.halo_lo = c->v.halo_lo; P.halo_hi = c->v.halo_hi;
  P.jet_lo = c->v.jet_lo; P.out_hi = c->v.out_hi;
  for (int side = 0; side < 2; ++side) {
    for (int k = 0; k < NF_MAX; ++k) P.nb[side].f[k] = c->nb_on[side] ? (T *)c->nb_fields[side][dst][k] : nullptr;
    P.nb_dz[side] = side == 0 ? c->nb_nz[0] : -c->v.L.nz;
  }
  P.jetD2 = c->p.jet_diameter * c->p.jet_diameter;
  P.jetU = (T)c->p.jet_velocity;
  P.jetP = (T)c->p.jet_perturbation;
  P.seed = c->p.seed;
  P.step_next = c->t + 1;
  P.step_ctr = nullptr;
  return P;
}

template <typename T>
int launch_generic(tslb_ctx *c, const StepParams<T> &P) {
  const Layout &L = P.L;
  const bool two = c->p.two_component != 0;
  if (two) {
    dim3 b(32, 8), g((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz + (P.halo_lo ? 1 : 0) + (P.halo_hi ? 1 : 0));
    phase_normals_kernel<T><<<g, b, 0, c->stream>>>(P);
    c->launches++;
  }
  dim3 b(32, 4), g((L.nx + 31) / 32, (L.ny + 3) / 4, L.nz);
  const int o3 = c->p.hermite_order >= 3;
  if (c->p.forcing == TSLB_FORCING_GUO) {
    dim3 bf(32, 8), gf((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz);
    force_kernel<T><<<gf, bf, 0, c->stream>>>(P);
    c->launches++;
    if (o3) generic_step_kernel<T, 3, true, true><<<g, b, 0, c->stream>>>(P);
    else generic_step_kernel<T, 2, true, true><<<g, b, 0, c->stream>>>(P);
  } else if (two) {
    if (o3) generic_step_kernel<T, 3, true><<<g, b, 0, c->stream>>>(P);
    else generic_step_kernel<T, 2, true><<<g, b, 0, c->stream>>>(P);
  } else {
    if (o3) generic_step_kernel<T, 3, false><<<g, b, 0, c->stream>>>(P);
    else generic_step_kernel<T, 2, false><<<g, b, 0, c->stream>>>(P);
  }
  c->launches++;
  CK(cudaGetLastError());
  return TSLB_OK;
}

__global__ void step_ctr_set_kernel(long long *ctr, long long v) { *ctr = v; }
__global__ void step_ctr_tick_kernel(long long *ctr) { *ctr += 1; }

// one time step src -> dst on the stream (no bookkeeping); step_ctr != null: graph capture
template <typename T>
int launch_step(tslb_ctx *c, int src, const long long *step_ctr) {
  StepParams<T> P = make_step_params<T>(c, src, src ^ 1);
  P.step_ctr = step_ctr;
  if (c->v.kernel == TSLB_KERNEL_TILED) {
    cudaError_t e = launch_tiled<T>(c->tiled, P, src, c->p.hermite_order, c->p.two_component != 0, c->stream);
    c->launches += (c->v.jet_lo || c->v.out_hi) ? 2 : 1;   // + the boundary-plane kernel with inflow/outflow
    return e == cudaSuccess ? TSLB_OK : c->cuda_fail(e, "launch_tiled");
  }
  return launch_generic<T>(c, P);
}

// Build (once per starting buffer) the graph of two steps cur -> cur^1 -> cur by stream capture.
template <typename T>
bool graph_build(tslb_ctx *c, int cur) {
  if (c->gexec[cur]) return true;
  if (c->graph_failed || !c->stream) return false;          // the legacy default stream cannot be captured
  if (!c->step_ctr && cudaMalloc((void **)&c->step_ctr, sizeof(long long)) != cudaSuccess) {
    cudaGetLastError();
    c->graph_failed = true;
    return false;
  }
  const long long keep = c->launches;
  cudaGraph_t g = nullptr;
  bool ok = cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (ok) {
    for (int h = 0; h < 2 && ok; ++h) {
      step_ctr_tick_kernel<<<1, 1, 0, c->stream>>>(c->step_ctr);
      ok = launch_step<T>(c, cur ^ h, c->step_ctr) == TSLB_OK;
    }
    ok = (cudaStreamEndCapture(c->stream, &g) == cudaSuccess) && ok && g;
  }
  if (ok) ok = cudaGraphInstantiate(&c->gexec[cur], g, 0) == cudaSuccess;
  if (g) cudaGraphDestroy(g);
  c->launches = keep;
  if (!ok) { cudaGetLastError(); c->gexec[cur] = nullptr; c->graph_failed = true; }
  return ok;
}

template <typename T>
int step_typed(tslb_ctx *c, int nsteps) {
  // one step launched from the host, with its bookkeeping
  auto one_step = [&]() -> int {
    int rc = launch_step<T>(c, c->cur, nullptr);
    if (rc != TSLB_OK) return rc;
    c->cur ^= 1;
    c->t++;
    if (c->stat_every && c->t % c->stat_every == 0) {
      const Layout &L = c->v.L;
      const size_t n = (size_t)L.nx * L.nz;
      dim3 b(128), g((L.nx + 127) / 128, L.nz);
      plane_stats_kernel<T><<<g, b, 0, c->stream>>>(L, c->p.two_component ? (const T *)c->fields[c->cur][F_PHI] : nullptr,
                                                   (const T *)c->fields[c->cur][F_UZ], (L.ny - 1) / 2, L.ny / 2, c->stat,
                                                   c->stat + n);
      CK(cudaGetLastError());
      c->launches++;
      c->stat_n++;
    }
    return TSLB_OK;
  };
  // Many short steps (small grids): replay a captured graph of two steps instead of launching 2-3 kernels per
  // step from the host.  Not for slabs (one step per call) nor while the mid-plane statistics are sampled.  The
  // first step of a context is launched directly (it sets the kernel attributes, which a capture must not).
  if (nsteps >= 5 && !c->v.slab && !c->stat_every && c->stream && !c->graph_failed) {
    if (c->launches == 0) {
      int rc = one_step();
      if (rc != TSLB_OK) return rc;
      --nsteps;
    }
    if (graph_build<T>(c, c->cur)) {
      const int pairs = nsteps / 2;
      const long long per_step = c->v.kernel == TSLB_KERNEL_TILED ? ((c->v.jet_lo || c->v.out_hi) ? 2 : 1)
                                 : (c->p.two_component ? (c->p.forcing == TSLB_FORCING_GUO ? 3 : 2) : 1);
      step_ctr_set_kernel<<<1, 1, 0, c->stream>>>(c->step_ctr, c->t);
      for (int g = 0; g < pairs; ++g) CK(cudaGraphLaunch(c->gexec[c->cur], c->stream));
      CK(cudaGetLastError());
      c->t += 2LL * pairs;
      c->launches += 2LL * pairs * (per_step + 1) + 1;      // + the one-thread counter kernels
      nsteps -= 2 * pairs;
    }
  }
  for (int s = 0; s < nsteps; ++s) {
    int rc = one_step();
    if (rc != TSLB_OK) return rc;
  }
  return TSLB_OK;
}

// tslb_get_physical_velocity: n of the phi that made the force into scratch, then one kernel
template <typename T>
int physvel_typed(tslb_ctx *c, void *const dst[3], int on_device) {
  const Layout &L = c->v.L;
  const size_t N = (size_t)L.nx * L.ny * L.nz;
  const bool guo = c->p.forcing == TSLB_FORCING_GUO;
  const bool use_force = c->p.two_component && (guo || c->t >= 1);
  // GUO: F of the current phi; KICK: F of the previous step's phi, still in the other buffer
  const int src = guo ? c->cur : c->cur ^ 1;
  StepParams<T> P = make_step_params<T>(c, src, src);
  for (int side = 0; side < 2; ++side)
    for (int k = 0; k < NF_MAX; ++k) P.nb[side].f[k] = nullptr;
  if (use_force) {
    if (!c->nrm[0]) {
      const size_t fb = round_up((size_t)L.field * sizeof(T), 256);
      if (!c->nrm_own) {
        cudaError_t e = cudaMalloc(&c->nrm_own, 3 * fb);
        if (e != cudaSuccess) return c->fail(TSLB_ENOMEM, "cudaMalloc(scratch normals): %s", cudaGetErrorString(e));
      }
      for (int k = 0; k < 3; ++k) P.nrm[k] = (T *)((char *)c->nrm_own + k * fb);
    }
    dim3 b(32, 8), g((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz);
    phase_normals_kernel<T><<<g, b, 0, c->stream>>>(P);
    CK(cudaGetLastError());
  }
  FieldSet<T> vel;
  for (int k = 0; k < NF_MAX; ++k) vel.f[k] = (T *)c->fields[c->cur][k];
  // host destinations: the three components go through scratch device memory of their own
  T *dev[3] = {nullptr, nullptr, nullptr};
  if (!on_device) {
    if (!c->pv_tmp) {
      cudaError_t e = cudaMalloc(&c->pv_tmp, 3 * N * sizeof(T));
      if (e != cudaSuccess) return c->fail(TSLB_ENOMEM, "cudaMalloc(physical velocity): %s", cudaGetErrorString(e));
    }
    T *tmp = (T *)c->pv_tmp;
    for (int a = 0; a < 3; ++a) dev[a] = dst[a] ? tmp + a * N : nullptr;
  } else {
    for (int a = 0; a < 3; ++a) dev[a] = (T *)dst[a];
  }
  dim3 b(32, 8), g((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz);
  physical_velocity_kernel<T><<<g, b, 0, c->stream>>>(P, vel, guo ? T(0.5) : T(-0.5), use_force ? 1 : 0, dev[0], dev[1], dev[2]);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess && !on_device)
    for (int a = 0; a < 3 && e == cudaSuccess; ++a)
      if (dst[a]) e = cudaMemcpyAsync(dst[a], dev[a], N * sizeof(T), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return c->cuda_fail(e, "tslb_get_physical_velocity");
  return TSLB_OK;
}

// staging for host pointers: two device buffers of one dense field each, a copy stream and the events that
// hand a buffer back and forth between the copy stream and the context's stream
int stage_setup(tslb_ctx *c) {
  const size_t N = (size_t)c->p.nx * c->p.ny * c->p.nz;
  for (int b = 0; b < 2; ++b) {
    if (!c->stage[b]) {
      cudaError_t e = cudaMalloc(&c->stage[b], N * c->v.esize);
      if (e != cudaSuccess) return c->fail(TSLB_ENOMEM, "cudaMalloc(stage): %s", cudaGetErrorString(e));
    }
    if (!c->ev_copied[b]) CK(cudaEventCreateWithFlags(&c->ev_copied[b], cudaEventDisableTiming));
    if (!c->ev_free[b]) CK(cudaEventCreateWithFlags(&c->ev_free[b], cudaEventDisableTiming));
  }
  if (!c->copy_stream) CK(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
  return TSLB_OK;
}

template <typename T>
int fill_all_ghosts(tslb_ctx *c, int buf) {
  const Layout &L = c->v.L;
  dim3 b(128), g((L.px + 127) / 128, L.py, L.nz);
  for (int k = 0; k < c->v.nfields; ++k) fill_ghosts_kernel<T><<<g, b, 0, c->stream>>>(L, (T *)c->fields[buf][k]);
  CK(cudaGetLastError());
  return TSLB_OK;
}

template <typename T>
int init_typed(tslb_ctx *c, const void *const src[NF_MAX], int on_device) {
  const Layout &L = c->v.L;
  const size_t N = (size_t)L.nx * L.ny * L.nz;
  dim3 b(128), g((L.nx + 127) / 128, L.ny, L.nz);
  // host arrays: field k is copied into one stage on the copy stream while the context's stream packs the
  // previous field out of the other stage
  if (!on_device) CK(cudaStreamSynchronize(c->stream));       // (the copy stream does not wait for earlier work)
  int nh = 0;
  for (int k = 0; k < c->v.nfields; ++k) {
    const T *d = nullptr;
    if (src[k]) {
      if (on_device) {
        d = (const T *)src[k];
      } else {
        const int sb = nh++ & 1;
        if (nh > 2) CK(cudaStreamWaitEvent(c->copy_stream, c->ev_free[sb], 0));
        CK(cudaMemcpyAsync(c->stage[sb], src[k], N * sizeof(T), cudaMemcpyHostToDevice, c->copy_stream));
        CK(cudaEventRecord(c->ev_copied[sb], c->copy_stream));
        CK(cudaStreamWaitEvent(c->stream, c->ev_copied[sb], 0));
        d = (const T *)c->stage[sb];
      }
    }
    pack_in_kernel<T><<<g, b, 0, c->stream>>>(L, d, (T *)c->fields[0][k], k == F_DRHO, d == nullptr);
    CK(cudaGetLastError());
    if (!on_device && src[k]) CK(cudaEventRecord(c->ev_free[(nh - 1) & 1], c->stream));
  }
  c->cur = 0;
  c->t = 0;
  if (c->v.jet_lo || c->v.out_hi) {
    StepParams<T> P = make_step_params<T>(c, 0, 0);
    dim3 gb((L.nx + 127) / 128, L.ny, 2);
    boundary_init_kernel<T><<<gb, b, 0, c->stream>>>(P, c->p.two_component);
    CK(cudaGetLastError());
  }
  int rc = fill_all_ghosts<T>(c, 0);
  if (rc != TSLB_OK) return rc;
  // the other buffer's ghosts/halo start from a defined state too
  const size_t zb = (size_t)L.gz * (size_t)L.plane * sizeof(T);
  for (int k = 0; k < c->v.nfields; ++k) {
    CK(cudaMemsetAsync((char *)c->fields[1][k] - zb, 0, (size_t)L.field * sizeof(T), c->stream));
    if (zb) {   // ghost planes of the current buffer: defined until the neighbours push theirs
      CK(cudaMemsetAsync((char *)c->fields[0][k] - zb, 0, zb, c->stream));
      CK(cudaMemsetAsync((char *)c->fields[0][k] + (size_t)L.plane * L.nz * sizeof(T), 0, zb, c->stream));
    }
  }
  CK(cudaStreamSynchronize(c->stream));
  return TSLB_OK;
}

template <typename T>
int get_typed(tslb_ctx *c, void *const dst[NF_MAX], int on_device) {
  const Layout &L = c->v.L;
  const size_t N = (size_t)L.nx * L.ny * L.nz;
  dim3 b(128), g((L.nx + 127) / 128, L.ny, L.nz);
  int nh = 0;
  for (int k = 0; k < c->v.nfields; ++k) {
    if (!dst[k]) continue;
    if (on_device) {
      pack_out_kernel<T><<<g, b, 0, c->stream>>>(L, (const T *)c->fields[c->cur][k], (T *)dst[k], k == F_DRHO);
      CK(cudaGetLastError());
      continue;
    }
    // host arrays: the context's stream unpacks field k into one stage while the copy stream sends the other out
    const int sb = nh++ & 1;
    if (nh > 2) CK(cudaStreamWaitEvent(c->stream, c->ev_free[sb], 0));
    pack_out_kernel<T><<<g, b, 0, c->stream>>>(L, (const T *)c->fields[c->cur][k], (T *)c->stage[sb], k == F_DRHO);
    CK(cudaGetLastError());
    CK(cudaEventRecord(c->ev_copied[sb], c->stream));
    CK(cudaStreamWaitEvent(c->copy_stream, c->ev_copied[sb], 0));
    CK(cudaMemcpyAsync(dst[k], c->stage[sb], N * sizeof(T), cudaMemcpyDeviceToHost, c->copy_stream));
    CK(cudaEventRecord(c->ev_free[sb], c->copy_stream));
  }
  if (nh) CK(cudaStreamSynchronize(c->copy_stream));
  CK(cudaStreamSynchronize(c->stream));
  return TSLB_OK;
}


// ---- tslb_get_physical_velocity_noalloc: scratch that nobody allocates.
// The three normal arrays n = grad(phi)/(|grad(phi)|+eps) of phase_normals_kernel live in ONE file-scope
// device array of a fixed, modest size: every GPU that loads the library holds it until the process
// exits.  In host code the array's NAME is only a stand-in, not a device address: a kernel given it
// would fault (or, where the GPU can reach host memory, silently use the wrong memory).  The device
// address comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr size_t NOALLOC_SCRATCH_BYTES = (size_t)12 << 20;   // 12 MiB: 3 arrays of <= 4 MiB each
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];
void *g_noalloc_ptr[TSLB_MAX_DEVICES] = {};                   // device address of the array, per device

// device must be the current device
cudaError_t noalloc_scratch_address(int device, void **out) {
  if (device < 0 || device >= TSLB_MAX_DEVICES) return cudaErrorInvalidDevice;
  if (!g_noalloc_ptr[device]) {
    void *ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[device] = ptr;
  }
  *out = g_noalloc_ptr[device];
  return cudaSuccess;
}

template <typename T>
int physvel_noalloc_typed(tslb_ctx *c, void *const dst[3], void *scratch) {
  const Layout &L = c->v.L;
  const bool guo = c->p.forcing == TSLB_FORCING_GUO;
  const bool use_force = c->p.two_component && (guo || c->t >= 1);
  // GUO: F of the current phi; KICK: F of the previous step's phi, still in the other buffer
  const int src = guo ? c->cur : c->cur ^ 1;
  StepParams<T> P = make_step_params<T>(c, src, src);
  for (int side = 0; side < 2; ++side)
    for (int k = 0; k < NF_MAX; ++k) P.nb[side].f[k] = nullptr;
  const size_t fb = round_up((size_t)L.field * sizeof(T), 256);
  for (int k = 0; k < 3; ++k) P.nrm[k] = (T *)((char *)scratch + k * fb);
  dim3 b(32, 8), g((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz);
  if (use_force) {
    // every entry of n that physical_velocity_kernel reads (the 27 neighbours of every node, by index
    // arithmetic: wrapped in x, y, wrapped or clamped in z) is written here first: nothing in the scratch
    // needs to start at zero, and the last call's contents are simply overwritten
    phase_normals_kernel<T><<<g, b, 0, c->stream>>>(P);
    CK(cudaGetLastError());
  }
  FieldSet<T> vel;
  for (int k = 0; k < NF_MAX; ++k) vel.f[k] = (T *)c->fields[c->cur][k];
  physical_velocity_kernel<T><<<g, b, 0, c->stream>>>(P, vel, guo ? T(0.5) : T(-0.5), use_force ? 1 : 0, (T *)dst[0],
                                                      (T *)dst[1], (T *)dst[2]);
  CK(cudaGetLastError());
  return TSLB_OK;
}

}  // namespace

// probe of the tiled kernel's reciprocal and square root (tslb_debug_math)
template <typename T>
__global__ void debug_math_kernel(int n, const double *in, double *orcp, double *osqrt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const T v = (T)in[i];
  orcp[i] = (double)tslb::rcp1(v);
  osqrt[i] = (double)tslb::sqrt1(v);
}

extern "C" {

size_t tslb_workspace_bytes(const tslb_params *p) {
  Validated v = validate(p);
  return v.ok ? v.bytes : 0;
}

int tslb_create(const tslb_params *p, tslb_ctx **out) {
  if (!out) { g_create_error = "out is NULL"; return TSLB_EINVAL; }
  *out = nullptr;
  Validated v = validate(p);
  if (!v.ok) { g_create_error = v.why; return TSLB_EINVAL; }
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    g_create_error = std::string("no CUDA device available (there is no CPU fallback): ") + cudaGetErrorString(e);
    return TSLB_ECUDA;
  }
  if (p->device < 0 || p->device >= ndev) { g_create_error = "device ordinal out of range"; return TSLB_EINVAL; }
  e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { g_create_error = std::string("cudaSetDevice: ") + cudaGetErrorString(e); return TSLB_ECUDA; }
  cudaDeviceProp prop;
  cudaGetDeviceProperties(&prop, p->device);
  if (prop.major != 10) {
    g_create_error = "this library is built for sm_100a (B200) only";
    return TSLB_ECUDA;
  }
  {
    // set-up of the allocation-free entry point: the device address of its scratch array, once per device
    // (a failure here is reported by tslb_get_physical_velocity_noalloc, which asks again)
    void *scratch = nullptr;
    if (noalloc_scratch_address(p->device, &scratch) != cudaSuccess) cudaGetLastError();
  }
  tslb_ctx *c = new (std::nothrow) tslb_ctx();
  if (!c) { g_create_error = "out of host memory"; return TSLB_ENOMEM; }
  c->p = *p;
  c->v = v;
  c->stream = (cudaStream_t)p->stream;
  if (p->workspace) {
    if (p->workspace_bytes < v.bytes || ((uintptr_t)p->workspace & 255)) {
      g_create_error = "workspace too small or not 256-byte aligned";
      delete c;
      return TSLB_EINVAL;
    }
    c->ws = p->workspace;
  } else {
    e = cudaMalloc(&c->ws, v.bytes);
    if (e != cudaSuccess) {
      g_create_error = std::string("cudaMalloc(workspace): ") + cudaGetErrorString(e);
      delete c;
      return TSLB_ENOMEM;
    }
    c->own_ws = true;
  }
  const size_t fb = round_up((size_t)v.L.field * v.esize, 256);
  char *base = (char *)c->ws;
  size_t off = 0;
  carve_fields(c->ws, v.L, v.esize, v.nfields, c->fields, &off);
  if (v.kernel == TSLB_KERNEL_GENERIC && p->two_component)
    for (int k = 0; k < 3; ++k) { c->nrm[k] = base + off + (size_t)v.L.gz * v.L.plane * v.esize; off += fb; }
  if (p->forcing == TSLB_FORCING_GUO)
    for (int k = 0; k < 3; ++k) { c->frc[k] = base + off; off += fb; }
  if (v.kernel == TSLB_KERNEL_TILED) {
    std::string why;
    if (!tiled_plan_create(c->tiled, p->precision, v.L, c->fields, v.nfields, p->device, why)) {
      g_create_error = "tiled kernel set-up failed: " + why;
      if (c->own_ws) cudaFree(c->ws);
      delete c;
      return TSLB_ECUDA;
    }
    c->kname = c->tiled.name;
  } else {
    c->kname = p->forcing == TSLB_FORCING_GUO ? "generic-guo" : "generic";
  }
  *out = c;
  return TSLB_OK;
}

int tslb_init_fields(tslb_ctx *c, const void *rho, const void *ux, const void *uy, const void *uz,
                     const void *phi, const void *const pineq[6], int pointers_on_device) {
  if (!c) return TSLB_EINVAL;
  if (!rho || !ux || !uy || !uz) return c->fail(TSLB_EINVAL, "rho, ux, uy, uz are required");
  if (c->p.two_component && !phi) return c->fail(TSLB_EINVAL, "phi is required when two_component");
  if (!c->p.two_component && phi) return c->fail(TSLB_EINVAL, "phi must be NULL when !two_component");
  CK(cudaSetDevice(c->p.device));
  if (!pointers_on_device) {
    int rc = stage_setup(c);
    if (rc != TSLB_OK) return rc;
  }
  const void *src[NF_MAX] = {rho, ux, uy, uz, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, phi};
  if (pineq)
    for (int k = 0; k < 6; ++k) src[F_PXX + k] = pineq[k];
  int rc = c->p.precision == TSLB_F32 ? init_typed<float>(c, src, pointers_on_device)
                                      : init_typed<double>(c, src, pointers_on_device);
  if (rc == TSLB_OK) c->inited = true;
  return rc;
}

int tslb_step(tslb_ctx *c, int nsteps) {
  if (!c) return TSLB_EINVAL;
  if (nsteps < 0) return c->fail(TSLB_EINVAL, "nsteps must be >= 0");
  if (!c->inited) return c->fail(TSLB_ESTATE, "tslb_step before tslb_init_fields");
  if (c->v.slab && nsteps > 1)
    return c->fail(TSLB_EINVAL, "a slab advances one step per call: its neighbours must finish step t before step t+1 starts");
  for (int side = 0; side < 2; ++side)
    if ((side == 0 ? c->v.halo_lo : c->v.halo_hi) && !c->nb_on[side] && nsteps > 0)
      return c->fail(TSLB_ESTATE, "halo face %d has no neighbour attached (tslb_attach_neighbor)", side);
  CK(cudaSetDevice(c->p.device));
  return c->p.precision == TSLB_F32 ? step_typed<float>(c, nsteps) : step_typed<double>(c, nsteps);
}

int tslb_get_moments(tslb_ctx *c, void *rho, void *ux, void *uy, void *uz, void *const pineq[6],
                     void *phi, int pointers_on_device) {
  if (!c) return TSLB_EINVAL;
  if (!c->inited) return c->fail(TSLB_ESTATE, "tslb_get_moments before tslb_init_fields");
  if (phi && !c->p.two_component) return c->fail(TSLB_EINVAL, "phi requested from a single-component context");
  CK(cudaSetDevice(c->p.device));
  if (!pointers_on_device) {
    int rc = stage_setup(c);
    if (rc != TSLB_OK) return rc;
  }
  void *dst[NF_MAX] = {rho, ux, uy, uz, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, phi};
  if (pineq)
    for (int k = 0; k < 6; ++k) dst[F_PXX + k] = pineq[k];
  return c->p.precision == TSLB_F32 ? get_typed<float>(c, dst, pointers_on_device)
                                    : get_typed<double>(c, dst, pointers_on_device);
}

int tslb_get_physical_velocity(tslb_ctx *c, void *ux, void *uy, void *uz, int pointers_on_device) {
  if (!c) return TSLB_EINVAL;
  if (!c->inited) return c->fail(TSLB_ESTATE, "tslb_get_physical_velocity before tslb_init_fields");
  if (c->v.slab) return c->fail(TSLB_EINVAL, "tslb_get_physical_velocity is not available on a z-slab");
  CK(cudaSetDevice(c->p.device));
  void *dst[3] = {ux, uy, uz};
  return c->p.precision == TSLB_F32 ? physvel_typed<float>(c, dst, pointers_on_device)
                                    : physvel_typed<double>(c, dst, pointers_on_device);
}

int tslb_get_physical_velocity_noalloc(tslb_ctx *c, void *ux, void *uy, void *uz) {
  if (!c) return TSLB_EINVAL;
  if (!c->inited) return c->fail(TSLB_ESTATE, "tslb_get_physical_velocity_noalloc before tslb_init_fields");
  if (c->v.slab) return c->fail(TSLB_EINVAL, "tslb_get_physical_velocity_noalloc is not available on a z-slab");
  const size_t need = 3 * round_up((size_t)c->v.L.field * c->v.esize, 256);
  if (need > NOALLOC_SCRATCH_BYTES)
    return c->fail(TSLB_EINVAL,
                   "tslb_get_physical_velocity_noalloc: the grid needs %zu bytes of scratch, the built-in array holds %zu "
                   "(use tslb_get_physical_velocity)", need, (size_t)NOALLOC_SCRATCH_BYTES);
  CK(cudaSetDevice(c->p.device));
  void *scratch = nullptr;
  cudaError_t e = noalloc_scratch_address(c->p.device, &scratch);
  if (e != cudaSuccess) return c->cuda_fail(e, "cudaGetSymbolAddress(scratch)");
  void *dst[3] = {ux, uy, uz};
  return c->p.precision == TSLB_F32 ? physvel_noalloc_typed<float>(c, dst, scratch)
                                    : physvel_noalloc_typed<double>(c, dst, scratch);
}

size_t tslb_noalloc_scratch_bytes(void) { return NOALLOC_SCRATCH_BYTES; }

void *tslb_workspace_ptr(const tslb_ctx *c) { return c ? c->ws : nullptr; }

int tslb_attach_neighbor(tslb_ctx *c, int face, void *nb_workspace, int nb_nz) {
  if (!c) return TSLB_EINVAL;
  if (face != 0 && face != 1) return c->fail(TSLB_EINVAL, "face must be 0 (z low) or 1 (z high)");
  if (!(face == 0 ? c->v.halo_lo : c->v.halo_hi)) return c->fail(TSLB_EINVAL, "face %d is not a TSLB_BC_HALO face", face);
  if (!nb_workspace || nb_nz < 2) return c->fail(TSLB_EINVAL, "neighbour workspace is NULL or its nz < 2");
  // a neighbour on another device of this process: map it (NVLink peer access)
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, nb_workspace) == cudaSuccess && at.type == cudaMemoryTypeDevice &&
      at.device != c->p.device) {
    CK(cudaSetDevice(c->p.device));
    cudaError_t e = cudaDeviceEnablePeerAccess(at.device, 0);
    if (e == cudaErrorPeerAccessAlreadyEnabled) { cudaGetLastError(); e = cudaSuccess; }
    if (e != cudaSuccess) return c->cuda_fail(e, "cudaDeviceEnablePeerAccess");
  } else {
    cudaGetLastError();
  }
  const Layout Ln = make_layout(c->p.nx, c->p.ny, nb_nz, GZ);
  carve_fields(nb_workspace, Ln, c->v.esize, c->v.nfields, c->nb_fields[face], nullptr);
  c->nb_nz[face] = nb_nz;
  c->nb_on[face] = true;
  return TSLB_OK;
}

int tslb_ipc_get_handle(tslb_ctx *c, void *handle64) {
  if (!c || !handle64) return TSLB_EINVAL;
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
  if (!c->own_ws) return c->fail(TSLB_ESTATE, "IPC export needs a workspace allocated by tslb_create");
  CK(cudaSetDevice(c->p.device));
  cudaIpcMemHandle_t h;
  CK(cudaIpcGetMemHandle(&h, c->ws));
  memcpy(handle64, &h, 64);
  return TSLB_OK;
}

int tslb_attach_neighbor_ipc(tslb_ctx *c, int face, const void *handle64, int nb_nz) {
  if (!c || !handle64) return TSLB_EINVAL;
  if (face != 0 && face != 1) return c->fail(TSLB_EINVAL, "face must be 0 (z low) or 1 (z high)");
  CK(cudaSetDevice(c->p.device));
  cudaIpcMemHandle_t h;
  memcpy(&h, handle64, 64);
  // two slabs with periodic z: both faces see the same neighbour -- open its handle once
  const int other = face ^ 1;
  if (c->nb_ipc[other] && memcmp(c->nb_handle[other], handle64, 64) == 0)
    return tslb_attach_neighbor(c, face, c->nb_ipc[other], nb_nz);
  void *base = nullptr;
  CK(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
  int rc = tslb_attach_neighbor(c, face, base, nb_nz);
  if (rc != TSLB_OK) { cudaIpcCloseMemHandle(base); return rc; }
  if (c->nb_ipc[face]) cudaIpcCloseMemHandle(c->nb_ipc[face]);
  c->nb_ipc[face] = base;
  memcpy(c->nb_handle[face], handle64, 64);
  return TSLB_OK;
}

int tslb_detach_neighbors(tslb_ctx *c) {
  if (!c) return TSLB_EINVAL;
  CK(cudaSetDevice(c->p.device));
  CK(cudaStreamSynchronize(c->stream));
  void *a = c->nb_ipc[0], *b = c->nb_ipc[1];
  if (a) CK(cudaIpcCloseMemHandle(a));
  if (b && b != a) CK(cudaIpcCloseMemHandle(b));
  c->nb_ipc[0] = c->nb_ipc[1] = nullptr;
  c->nb_on[0] = c->nb_on[1] = false;
  return TSLB_OK;
}

int tslb_halo_push(tslb_ctx *c) {
  if (!c) return TSLB_EINVAL;
  if (!c->inited) return c->fail(TSLB_ESTATE, "tslb_halo_push before tslb_init_fields");
  CK(cudaSetDevice(c->p.device));
  const Layout &L = c->v.L;
  const size_t pb = (size_t)L.plane * c->v.esize;
  for (int side = 0; side < 2; ++side) {
    if (!c->nb_on[side]) continue;
    for (int k = 0; k < c->v.nfields; ++k) {
      // my planes 0,1 -> the lower neighbour's planes nz', nz'+1; my planes nz-2, nz-1 -> the upper
      // neighbour's planes -2, -1 (padded planes are contiguous, ghost columns included)
      const char *src = (const char *)c->fields[c->cur][k] + (side == 0 ? 0 : (size_t)(L.nz - 2) * pb);
      char *dst = (char *)c->nb_fields[side][c->cur][k];
      if (side == 0) dst += (size_t)c->nb_nz[0] * pb; else dst -= 2 * pb;
      CK(cudaMemcpyAsync(dst, src, 2 * pb, cudaMemcpyDefault, c->stream));
    }
  }
  return TSLB_OK;
}

int tslb_stats_begin(tslb_ctx *c, int every) {
  if (!c) return TSLB_EINVAL;
  if (every < 1) return c->fail(TSLB_EINVAL, "every must be >= 1");
  CK(cudaSetDevice(c->p.device));
  const size_t n = (size_t)c->p.nx * c->p.nz;
  if (!c->stat) {
    cudaError_t e = cudaMalloc((void **)&c->stat, 2 * n * sizeof(double));
    if (e != cudaSuccess) return c->fail(TSLB_ENOMEM, "cudaMalloc(stats): %s", cudaGetErrorString(e));
  }
  CK(cudaMemsetAsync(c->stat, 0, 2 * n * sizeof(double), c->stream));
  c->stat_every = every;
  c->stat_n = 0;
  return TSLB_OK;
}

int tslb_stats_get(tslb_ctx *c, double *sum_phi, double *sum_uz, long long *nsamples) {
  if (!c) return TSLB_EINVAL;
  if (!c->stat) return c->fail(TSLB_ESTATE, "tslb_stats_get before tslb_stats_begin");
  CK(cudaSetDevice(c->p.device));
  const size_t n = (size_t)c->p.nx * c->p.nz;
  if (sum_phi) CK(cudaMemcpyAsync(sum_phi, c->stat, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  if (sum_uz) CK(cudaMemcpyAsync(sum_uz, c->stat + n, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if (nsamples) *nsamples = c->stat_n;
  return TSLB_OK;
}

int tslb_stats_end(tslb_ctx *c) {
  if (!c) return TSLB_EINVAL;
  c->stat_every = 0;
  return TSLB_OK;
}

long long tslb_step_count(const tslb_ctx *c) { return c ? c->t : -1; }
const char *tslb_kernel_name(const tslb_ctx *c) { return c ? c->kname.c_str() : ""; }
long long tslb_launch_count(const tslb_ctx *c) { return c ? c->launches : -1; }

int tslb_debug_xi(tslb_ctx *c, long long step, double *out_host) {
  if (!c || !out_host) return TSLB_EINVAL;
  CK(cudaSetDevice(c->p.device));
  const int nx = c->p.nx, ny = c->p.ny;
  double *d = nullptr;
  CK(cudaMalloc(&d, sizeof(double) * nx * ny));
  dim3 b(128), g((nx + 127) / 128, ny);
  if (c->p.precision == TSLB_F32) debug_xi_kernel<float><<<g, b, 0, c->stream>>>(c->p.seed, nx, ny, step, d);
  else debug_xi_kernel<double><<<g, b, 0, c->stream>>>(c->p.seed, nx, ny, step, d);
  cudaError_t e = cudaMemcpyAsync(out_host, d, sizeof(double) * nx * ny, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(d);
  if (e != cudaSuccess) return c->cuda_fail(e, "tslb_debug_xi");
  return TSLB_OK;
}

int tslb_debug_math(tslb_ctx *c, int n, const double *in_host, double *out_rcp_host, double *out_sqrt_host) {
  if (!c || !in_host || !out_rcp_host || !out_sqrt_host || n < 1) return TSLB_EINVAL;
  CK(cudaSetDevice(c->p.device));
  double *d = nullptr;
  CK(cudaMalloc(&d, sizeof(double) * 3 * (size_t)n));
  cudaError_t e = cudaMemcpyAsync(d, in_host, sizeof(double) * n, cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess) {
    if (c->p.precision == TSLB_F32) debug_math_kernel<float><<<(n + 127) / 128, 128, 0, c->stream>>>(n, d, d + n, d + 2 * (size_t)n);
    else debug_math_kernel<double><<<(n + 127) / 128, 128, 0, c->stream>>>(n, d, d + n, d + 2 * (size_t)n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(out_rcp_host, d + n, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(out_sqrt_host, d + 2 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(d);
  if (e != cudaSuccess) return c->cuda_fail(e, "tslb_debug_math");
  return TSLB_OK;
}

int tslb_destroy(tslb_ctx *c) {
  if (!c) return TSLB_OK;
  cudaSetDevice(c->p.device);
  cudaStreamSynchronize(c->stream);
  tiled_plan_destroy(c->tiled);
  for (int side = 0; side < 2; ++side)
    if (c->nb_ipc[side]) cudaIpcCloseMemHandle(c->nb_ipc[side]);
  for (int g = 0; g < 2; ++g)
    if (c->gexec[g]) cudaGraphExecDestroy(c->gexec[g]);
  if (c->step_ctr) cudaFree(c->step_ctr);
  for (int b = 0; b < 2; ++b) {
    if (c->stage[b]) cudaFree(c->stage[b]);
    if (c->ev_copied[b]) cudaEventDestroy(c->ev_copied[b]);
    if (c->ev_free[b]) cudaEventDestroy(c->ev_free[b]);
  }
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->pv_tmp) cudaFree(c->pv_tmp);
  if (c->stat) cudaFree(c->stat);
  if (c->nrm_own) cudaFree(c->nrm_own);
  if (c->own_ws && c->ws) cudaFree(c->ws);
  delete c;
  return TSLB_OK;
}

const char *tslb_last_error(const tslb_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
