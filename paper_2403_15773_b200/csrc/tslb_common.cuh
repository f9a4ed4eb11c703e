// tslb_common.cuh -- device-side data layout and small helpers shared by the TSLB kernels.
//
// Internal HBM layout.  Every field is one SoA array in a PADDED layout
//   element (x,y,z)  ->  ((z * py) + (y + GY)) * px + (x + GX),   px = nx + 2 GX, py = ny + 2 GY
// with GX = 8 ghost columns and GY = 2 ghost rows on each side that mirror the periodic image
// (x and y are always periodic).  Ghosts let a TMA box that starts at x0-2 / y0-2 never leave
// the tensor and keep every interior row 32-byte (sector) aligned.  z has no ghosts on a single
// GPU: planes are fetched one at a time and the plane index is wrapped (periodic) or clamped
// (inflow/outflow).  A z-SLAB of a multi-GPU run stores gz = 2 extra
// planes below z = 0 and above z = nz-1; the field pointers handed to the kernels point at plane 0,
// so idx() is valid for z in [-gz, nz+gz).  The slab's neighbours write those planes (their two face
// planes of phi, one of the moments) from inside their own step kernel through peer pointers.
//
// Field order: 0 drho (= rho - 1, note N1), 1..3 u, 4..9 Pi^neq (xx,yy,zz,xy,xz,yz), 10 phi.
#pragma once
#include <cstddef>
#include <cstdint>

namespace tslb {

constexpr int GX = 8;
constexpr int GY = 2;
constexpr int GZ = 2;      // ghost planes per z face of a slab
constexpr int NF_FLOW = 10;
constexpr int NF_MAX = 11;
enum Field { F_DRHO = 0, F_UX, F_UY, F_UZ, F_PXX, F_PYY, F_PZZ, F_PXY, F_PXZ, F_PYZ, F_PHI };

struct Layout {
  int nx, ny, nz;
  int px, py;            // padded row length / rows per plane
  int gz;                // ghost planes on each side of z (0, or GZ in slab mode)
  long long plane;       // px * py
  long long field;       // elements per field array (plane * (nz + 2 gz), rounded up to 64 elements)
  __host__ __device__ inline long long idx(int x, int y, int z) const {
    return ((long long)z * py + (y + GY)) * px + (x + GX);
  }
};

template <typename T>
struct FieldSet {
  T *f[NF_MAX];
};

// Parameters common to all step kernels (passed by value as a __grid_constant__).
template <typename T>
struct StepParams {
  Layout L;
  FieldSet<T> in, out;   // time t (read only) and time t+1 (written)
  T *nrm[3];             // generic path only: scratch n = grad(phi)/(|grad(phi)|+eps), dense padded
  T *frc[3];             // TSLB_FORCING_GUO only: scratch F = sigma kappa grad(phi) of the time-t phi
  T omc;                 // 1 - omega                               (eq. 5)
  T sigma;               // surface tension                         (eq. 20)
  T gamma;               // anti-diffusion 2/W                      (eq. 24, A8)
  int zper;              // 1: z periodic (wrap); 0: clamp, unless the face is a halo face
  int halo_lo, halo_hi;  // slab faces: planes z < 0 / z >= nz are ghost planes filled by the neighbour
  int jet_lo, out_hi;    // plane 0 is the jet inflow plane / plane nz-1 the outflow plane (O9)
  // halo push: the neighbour slabs' TIME t+1 buffers (same nx, ny, layout), or null.  My plane j is
  // the neighbour's plane j + nb_dz[side]: side 0 (below me): nz_of_that_slab + j for j = 0, 1;
  // side 1 (above me): j - nz for j = nz-2, nz-1.  phi: both planes; moments: the face plane only.
  FieldSet<T> nb[2];
  int nb_dz[2];
  // jet inflow (A10, A12)
  double jetD2;          // D^2, compared with (2x-(nx-1))^2 + (2y-(ny-1))^2
  T jetU, jetP;
  unsigned long long seed;
  long long step_next;   // index t+1 of the step being computed (keys the hash) ...
  const long long *step_ctr;   // ... or, when not null (replayed CUDA graph), where to read it on the device
};

// Counter-based inflow perturbation (reading A12): splitmix64 finaliser of
// seed + (counter+1)*golden, counter = step*nx*ny + x + nx*y; top 24 bits k ->
// xi = (2k + 1 - 2^24) * 2^-24, formed from the integer numerator so the conversion is exact in
// fp32 and fp64.
__host__ __device__ inline int xi_numerator(unsigned long long seed, int x, int y, int nx, int ny,
                                            long long step) {
  unsigned long long counter =
      (unsigned long long)step * ((unsigned long long)nx * (unsigned long long)ny) +
      (unsigned long long)(x + nx * y);
  unsigned long long z = seed + (counter + 1ULL) * 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  z = z ^ (z >> 31);
  long long k = (long long)(z >> 40);
  return (int)(2 * k + 1 - (1LL << 24));
}

template <typename T>
__host__ __device__ inline T xi_value(unsigned long long seed, int x, int y, int nx, int ny, long long step) {
  return (T)xi_numerator(seed, x, y, nx, ny, step) * (T)(1.0 / 16777216.0);
}

// index t+1 of the step being computed
template <typename T>
__device__ __forceinline__ long long step_index(const StepParams<T> &P) { return P.step_ctr ? *P.step_ctr : P.step_next; }

// source plane for a read at z, at most two planes outside [0, nz): ghost plane of a slab face,
// periodic image, or the clamped boundary plane.  Branch-free: it sits in the hot loop of the tiled
// kernel, whose body is at the instruction-cache limit.
template <typename T>
__host__ __device__ inline int zsrc(const StepParams<T> &P, int z) {
  const int nz = P.L.nz;
  const int lo = P.halo_lo ? z : (P.zper ? (nz == 1 ? 0 : z + nz) : 0);
  const int hi = P.halo_hi ? z : (P.zper ? (nz == 1 ? 0 : z - nz) : nz - 1);
  return z < 0 ? lo : (z >= nz ? hi : z);
}

__host__ __device__ inline bool in_nozzle(int x, int y, int nx, int ny, double D2) {
  long long ix = 2LL * x - (nx - 1), iy = 2LL * y - (ny - 1);
  return (double)(ix * ix + iy * iy) < D2;
}

}  // namespace tslb
