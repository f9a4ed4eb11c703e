// tslb_generic.cuh -- reference-quality CUDA path: one thread per node, direct global loads.
//
// Works for any grid size and both boundary types; it is the kernel the tiled path is checked
// against and the fallback for grids that are not multiples of the tile.  Two launches per step
// when two_component: (1) phase_normals: n = G/(|G|+eps) from the OLD phi into scratch,
// (2) generic_step: everything else.  Periodic wrap / z clamp by index arithmetic (ghost cells
// are not read here).
#pragma once
#include "tslb_math.cuh"

namespace tslb {

__device__ __forceinline__ int wrapi(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

template <typename T> __device__ __forceinline__ T eps_n() { return T(1e-12); }
template <typename T> __device__ __forceinline__ T tsqrt(T x);
template <> __device__ __forceinline__ float tsqrt<float>(float x) { return sqrtf(x); }
template <> __device__ __forceinline__ double tsqrt<double>(double x) { return sqrt(x); }

// G = (1/c_s^2) sum_i w_i c_i phi(x + c_i)  (eqs. 20-21, readings A6/A7) in
// its separable form: central difference along one axis, [1/6,2/3,1/6] along the other two.
template <typename T>
__device__ __forceinline__ void grad_phi(const T *__restrict__ phi, const StepParams<T> &P, int x, int y, int z,
                                         T G[3]) {
  const Layout &L = P.L;
  T gx = 0, gy = 0, gz = 0;
#pragma unroll
  for (int dz = -1; dz <= 1; ++dz) {
    const int zz = zsrc(P, z + dz);
#pragma unroll
    for (int dy = -1; dy <= 1; ++dy) {
      const int yy = wrapi(y + dy, L.ny);
#pragma unroll
      for (int dx = -1; dx <= 1; ++dx) {
        const int xx = wrapi(x + dx, L.nx);
        const T w = w1d<T>(dx) * w1d<T>(dy) * w1d<T>(dz) * T(3);
        const T p = phi[L.idx(xx, yy, zz)];
        gx += (w * T(dx)) * p;
        gy += (w * T(dy)) * p;
        gz += (w * T(dz)) * p;
      }
    }
  }
  G[0] = gx; G[1] = gy; G[2] = gz;
}

// kappa = -(1/c_s^2) sum_i w_i c_i . n(x + c_i) from the scratch normals   (eq. 21, A6)
template <typename T>
__device__ __forceinline__ T kappa_at(const StepParams<T> &P, int x, int y, int z) {
  const Layout &L = P.L;
  T div = T(0);
#pragma unroll
  for (int dz = -1; dz <= 1; ++dz) {
    const int zz = zsrc(P, z + dz);
#pragma unroll
    for (int dy = -1; dy <= 1; ++dy) {
      const int yy = wrapi(y + dy, L.ny);
#pragma unroll
      for (int dx = -1; dx <= 1; ++dx) {
        if (dx == 0 && dy == 0 && dz == 0) continue;
        const int xx = wrapi(x + dx, L.nx);
        const long long j = L.idx(xx, yy, zz);
        const T w = w1d<T>(dx) * w1d<T>(dy) * w1d<T>(dz) * T(3);
        if (dx != 0) div += (w * T(dx)) * P.nrm[0][j];
        if (dy != 0) div += (w * T(dy)) * P.nrm[1][j];
        if (dz != 0) div += (w * T(dz)) * P.nrm[2][j];
      }
    }
  }
  return -div;
}

template <typename T>
__global__ void __launch_bounds__(256) phase_normals_kernel(const __grid_constant__ StepParams<T> P) {
  const Layout &L = P.L;
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = (int)blockIdx.z - (P.halo_lo ? 1 : 0);   // slab: n is needed on one ghost plane per halo face
  if (x >= L.nx || y >= L.ny) return;
  T G[3];
  grad_phi<T>(P.in.f[F_PHI], P, x, y, z, G);
  const T mag = tsqrt<T>(G[0] * G[0] + G[1] * G[1] + G[2] * G[2]);
  const T inv = T(1) / (mag + eps_n<T>());
  const long long i = L.idx(x, y, z);
  P.nrm[0][i] = G[0] * inv;
  P.nrm[1][i] = G[1] * inv;
  P.nrm[2][i] = G[2] * inv;
}

// Imposed moments on the two z boundary planes (eqs. 9-10; A10, A11): all
// neighbour values are OLD (time-t) values of the plane next to the boundary.
template <typename T>
__device__ __forceinline__ void boundary_node(const StepParams<T> &P, const FieldSet<T> &src, int x, int y,
                                              int z, long long step_index, T out[NF_MAX], bool two) {
  const Layout &L = P.L;
  if (z == 0) {
    const long long f = L.idx(x, y, 1);
    const bool inside = in_nozzle(x, y, L.nx, L.ny, P.jetD2);
    out[F_DRHO] = src.f[F_DRHO][f];
    out[F_UX] = T(0);
    out[F_UY] = T(0);
    out[F_UZ] = inside ? P.jetU * (T(1) + P.jetP * xi_value<T>(P.seed, x, y, L.nx, L.ny, step_index)) : T(0);
#pragma unroll
    for (int k = F_PXX; k <= F_PYZ; ++k) out[k] = src.f[k][f];
    out[F_PHI] = inside ? T(1) : T(0);
  } else {
    const long long f = L.idx(x, y, L.nz - 2);
    out[F_DRHO] = T(0);
#pragma unroll
    for (int k = F_UX; k <= F_PYZ; ++k) out[k] = src.f[k][f];
    out[F_PHI] = two ? src.f[F_PHI][f] : T(0);
  }
}

// F = sigma kappa G of the time-t phi into the scratch arrays frc (TSLB_FORCING_GUO), zero on the
// inflow/outflow planes (their moments are imposed, O9).  Needs phase_normals_kernel first.
template <typename T>
__global__ void __launch_bounds__(256) force_kernel(const __grid_constant__ StepParams<T> P) {
  const Layout &L = P.L;
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= L.nx || y >= L.ny) return;
  T s = T(0), G[3] = {T(0), T(0), T(0)};
  if (!((P.jet_lo && z == 0) || (P.out_hi && z == L.nz - 1))) {
    grad_phi<T>(P.in.f[F_PHI], P, x, y, z, G);
    s = P.sigma * kappa_at<T>(P, x, y, z);
  }
  const long long i = L.idx(x, y, z);
  P.frc[0][i] = s * G[0];
  P.frc[1][i] = s * G[1];
  P.frc[2][i] = s * G[2];
}

// Time-centred velocity (include/tslb.h tslb_get_physical_velocity) into dense arrays: the stored
// velocity of `vel` plus sgn * F / rho, F = sigma kappa G of the phi in P.in (needs
// phase_normals_kernel on the same P first); F = 0 on inflow/outflow planes and when !use_force.
template <typename T>
__global__ void __launch_bounds__(256) physical_velocity_kernel(const __grid_constant__ StepParams<T> P, FieldSet<T> vel,
                                                                T sgn, int use_force, T *dx_, T *dy_, T *dz_) {
  const Layout &L = P.L;
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= L.nx || y >= L.ny) return;
  T s = T(0), G[3] = {T(0), T(0), T(0)};
  const long long i = L.idx(x, y, z);
  if (use_force && !((P.jet_lo && z == 0) || (P.out_hi && z == L.nz - 1))) {
    grad_phi<T>(P.in.f[F_PHI], P, x, y, z, G);
    s = sgn * P.sigma * kappa_at<T>(P, x, y, z) / (T(1) + vel.f[F_DRHO][i]);
  }
  const long long o = (long long)x + (long long)L.nx * (y + (long long)L.ny * z);
  if (dx_) dx_[o] = vel.f[F_UX][i] + s * G[0];
  if (dy_) dy_[o] = vel.f[F_UY][i] + s * G[1];
  if (dz_) dz_[o] = vel.f[F_UZ][i] + s * G[2];
}

template <typename T, int ORDER, bool TWO, bool GUO = false>
__global__ void __launch_bounds__(128) generic_step_kernel(const __grid_constant__ StepParams<T> P) {
  const Layout &L = P.L;
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= L.nx || y >= L.ny) return;
  const long long i0 = L.idx(x, y, z);
  constexpr int NF = TWO ? 11 : 10;

  if ((P.jet_lo && z == 0) || (P.out_hi && z == L.nz - 1)) {
    T o[NF_MAX];
    boundary_node<T>(P, P.in, x, y, z, step_index(P), o, TWO);
#pragma unroll
    for (int k = 0; k < NF; ++k) P.out.f[k][i0] = o[k];
    return;
  }

  // a1-a4: pull the 27 neighbours' moments, rebuild f_i^post(x - c_i), accumulate the Hermite
  // moments of the streamed populations (eq. 6, 79).
  T M[10];
#pragma unroll
  for (int k = 0; k < 10; ++k) M[k] = T(0);
#pragma unroll
  for (int cz = -1; cz <= 1; ++cz) {
    const int zz = zsrc(P, z - cz);
#pragma unroll
    for (int cy = -1; cy <= 1; ++cy) {
      const int yy = wrapi(y - cy, L.ny);
#pragma unroll
      for (int cx = -1; cx <= 1; ++cx) {
        const int xx = wrapi(x - cx, L.nx);
        const long long j = L.idx(xx, yy, zz);
        T Kt[NK];
        if (GUO)
          post_collision_coeffs_guo<ORDER, T>(P.in.f[F_DRHO][j], P.in.f[F_UX][j], P.in.f[F_UY][j], P.in.f[F_UZ][j],
                                              P.in.f[F_PXX][j], P.in.f[F_PYY][j], P.in.f[F_PZZ][j], P.in.f[F_PXY][j],
                                              P.in.f[F_PXZ][j], P.in.f[F_PYZ][j], P.frc[0][j], P.frc[1][j], P.frc[2][j],
                                              P.omc, Kt);
        else
          post_collision_coeffs<ORDER, T>(P.in.f[F_DRHO][j], P.in.f[F_UX][j], P.in.f[F_UY][j], P.in.f[F_UZ][j],
                                          P.in.f[F_PXX][j], P.in.f[F_PYY][j], P.in.f[F_PZZ][j], P.in.f[F_PXY][j],
                                          P.in.f[F_PXZ][j], P.in.f[F_PYZ][j], P.omc, Kt);
        const T x1 = h1d<T>(1, cx), x2 = h1d<T>(2, cx);
        const T y1 = h1d<T>(1, cy), y2 = h1d<T>(2, cy);
        const T z1 = h1d<T>(1, cz), z2 = h1d<T>(2, cz);
        T s = Kt[K000] + Kt[K100] * x1 + Kt[K010] * y1 + Kt[K001] * z1 + Kt[K200] * x2 + Kt[K020] * y2 +
              Kt[K002] * z2 + Kt[K110] * (x1 * y1) + Kt[K101] * (x1 * z1) + Kt[K011] * (y1 * z1);
        if (ORDER >= 3)
          s += Kt[K210] * (x2 * y1) + Kt[K201] * (x2 * z1) + Kt[K120] * (x1 * y2) + Kt[K021] * (y2 * z1) +
               Kt[K102] * (x1 * z2) + Kt[K012] * (y1 * z2) + Kt[K111] * (x1 * y1 * z1);
        const T f = (w1d<T>(cx) * w1d<T>(cy) * w1d<T>(cz)) * s;   // f_i^post(x - c_i) - w_i
        M[0] += f;
        M[1] += x1 * f; M[2] += y1 * f; M[3] += z1 * f;
        M[4] += x2 * f; M[5] += y2 * f; M[6] += z2 * f;
        M[7] += (x1 * y1) * f; M[8] += (x1 * z1) * f; M[9] += (y1 * z1) * f;
      }
    }
  }
  T drho, ub[3], pin[6];
  finish_moments<T>(M, drho, ub, pin);

  T phin = T(0);
  if (TWO) {
    if (!GUO) {
      // a5: G at the node from the OLD phi; kappa = -(1/c_s^2) sum_i w_i c_i . n(x + c_i)
      T G[3];
      grad_phi<T>(P.in.f[F_PHI], P, x, y, z, G);
      const T kappa = kappa_at<T>(P, x, y, z);
      // a6: kick u' = u_b + F / rho', F = sigma kappa G   (A9)
      const T s = P.sigma * kappa / (T(1) + drho);
      ub[0] += s * G[0]; ub[1] += s * G[1]; ub[2] += s * G[2];
    }
    // a7: phi'(x) = sum_{i in D3Q7} w_i [ phi (1 + c_i.u / c_sg^2) + gamma phi (1-phi) c_i.n ](x - c_i)
    const T *phi = P.in.f[F_PHI];
    const T pc = phi[i0];
    T acc = T(0.25) * pc;
    const int xm = wrapi(x - 1, L.nx), xp = wrapi(x + 1, L.nx);
    const int ym = wrapi(y - 1, L.ny), yp = wrapi(y + 1, L.ny);
    const int zm = zsrc(P, z - 1), zp = zsrc(P, z + 1);
    const long long jn[6] = {L.idx(xm, y, z), L.idx(xp, y, z), L.idx(x, ym, z),
                             L.idx(x, yp, z), L.idx(x, y, zm), L.idx(x, y, zp)};
    // neighbour at x - c_i: c_i = +e for the "minus" neighbour, -e for the "plus" neighbour
    const int comp[6] = {0, 0, 1, 1, 2, 2};
    const T sgn[6] = {T(1), T(-1), T(1), T(-1), T(1), T(-1)};
#pragma unroll
    for (int q = 0; q < 6; ++q) {
      const T p = phi[jn[q]];
      T uc = P.in.f[F_UX + comp[q]][jn[q]];
      // A18: phi is advected with the time-centred velocity u_b + F/(2 rho) of the source node
      if (GUO) uc += P.frc[comp[q]][jn[q]] / (T(2) * (T(1) + P.in.f[F_DRHO][jn[q]]));
      const T nc = P.nrm[comp[q]][jn[q]];
      acc += T(0.125) * (p * (T(1) + sgn[q] * T(4) * uc) + P.gamma * p * (T(1) - p) * (sgn[q] * nc));
    }
    phin = acc;
  }

  P.out.f[F_DRHO][i0] = drho;
  P.out.f[F_UX][i0] = ub[0];
  P.out.f[F_UY][i0] = ub[1];
  P.out.f[F_UZ][i0] = ub[2];
#pragma unroll
  for (int k = 0; k < 6; ++k) P.out.f[F_PXX + k][i0] = pin[k];
  if (TWO) P.out.f[F_PHI][i0] = phin;
  // halo push into the neighbour slabs' ghost planes (interior nodes; this path never reads ghost
  // columns).  Slab face planes that are jet boundary planes have no neighbour.
#pragma unroll
  for (int side = 0; side < 2; ++side) {
    if (!P.nb[side].f[0]) continue;
    const int depth = side == 0 ? z : L.nz - 1 - z;     // 0: face plane, 1: the plane behind it
    if (depth > 1) continue;
    const long long i1 = L.idx(x, y, z + P.nb_dz[side]);
    if (depth == 0) {
      P.nb[side].f[F_DRHO][i1] = drho;
      P.nb[side].f[F_UX][i1] = ub[0];
      P.nb[side].f[F_UY][i1] = ub[1];
      P.nb[side].f[F_UZ][i1] = ub[2];
#pragma unroll
      for (int k = 0; k < 6; ++k) P.nb[side].f[F_PXX + k][i1] = pin[k];
    }
    if (TWO) P.nb[side].f[F_PHI][i1] = phin;
  }
}

// ---- layout conversion / ghost maintenance / boundary init -------------------------------

// dense user array -> padded internal field (interior only); sub1: store value - 1 (rho -> drho)
template <typename T>
__global__ void pack_in_kernel(Layout L, const T *__restrict__ src, T *__restrict__ dst, int sub1, int zero) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y;
  const int z = blockIdx.z;
  if (x >= L.nx) return;
  T v = zero ? T(0) : src[(long long)x + (long long)L.nx * (y + (long long)L.ny * z)];
  if (sub1) v -= T(1);
  dst[L.idx(x, y, z)] = v;
}

template <typename T>
__global__ void pack_out_kernel(Layout L, const T *__restrict__ src, T *__restrict__ dst, int add1) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y;
  const int z = blockIdx.z;
  if (x >= L.nx) return;
  T v = src[L.idx(x, y, z)];
  if (add1) v += T(1);
  dst[(long long)x + (long long)L.nx * (y + (long long)L.ny * z)] = v;
}

// refresh the periodic ghost columns/rows of one field from its interior
template <typename T>
__global__ void fill_ghosts_kernel(Layout L, T *__restrict__ a) {
  const int X = blockIdx.x * blockDim.x + threadIdx.x;   // padded coordinates
  const int Y = blockIdx.y;
  const int z = blockIdx.z;
  if (X >= L.px) return;
  const int x = X - GX, y = Y - GY;
  if (x >= 0 && x < L.nx && y >= 0 && y < L.ny) return;
  const int xs = ((x % L.nx) + L.nx) % L.nx, ys = ((y % L.ny) + L.ny) % L.ny;
  a[((long long)z * L.py + Y) * L.px + X] = a[L.idx(xs, ys, z)];
}

// O9 applied in place to the initial fields (hash step index 0)
template <typename T>
__global__ void boundary_init_kernel(const __grid_constant__ StepParams<T> P, int two) {
  const Layout &L = P.L;
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y;
  const int z = blockIdx.z ? L.nz - 1 : 0;
  if (x >= L.nx) return;
  if (blockIdx.z ? !P.out_hi : !P.jet_lo) return;
  T o[NF_MAX];
  boundary_node<T>(P, P.out, x, y, z, 0, o, two != 0);
  const long long i0 = L.idx(x, y, z);
  const int nf = two ? 11 : 10;
  for (int k = 0; k < nf; ++k) P.out.f[k][i0] = o[k];
}

// Running sums for the time averages <phi>, <u_z> on the mid x-z plane (Figs. 5-6;
// SURVEY NEXT-3).  The jet axis is at y = (ny-1)/2: rows y0 = floor, y1 = ceil of it are averaged.
// One thread per (x, z); fp64 accumulators; traffic 2 rows per plane, negligible beside the step.
template <typename T>
__global__ void plane_stats_kernel(Layout L, const T *__restrict__ phi, const T *__restrict__ uz, int y0, int y1,
                                   double *__restrict__ sum_phi, double *__restrict__ sum_uz) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int z = blockIdx.y;
  if (x >= L.nx) return;
  const long long i0 = L.idx(x, y0, z), i1 = L.idx(x, y1, z);
  const long long o = (long long)z * L.nx + x;
  sum_uz[o] += 0.5 * ((double)uz[i0] + (double)uz[i1]);
  if (phi) sum_phi[o] += 0.5 * ((double)phi[i0] + (double)phi[i1]);
}

template <typename T>
__global__ void debug_xi_kernel(unsigned long long seed, int nx, int ny, long long step, double *out) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y;
  if (x >= nx) return;
  out[x + nx * y] = (double)xi_value<T>(seed, x, y, nx, ny, step);
}

}  // namespace tslb
