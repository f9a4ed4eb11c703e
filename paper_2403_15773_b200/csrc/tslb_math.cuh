// tslb_math.cuh -- per-node algebra of the TSLB step in the tensor-product Hermite basis.
//
// D3Q27 is the tensor product of three D1Q3 lattices: c in {-1,0,1}, w(0)=2/3, w(+-1)=1/6,
// c_s^2 = 1/3 (reading A1).  In the 1-D basis h0 = 1, h1 = c, h2 = c^2 - 1/3
// (norms 1, 1/3, 2/9) the post-collision populations of PAPER.md:91 eq. 5 with the third-order
// expansions of PAPER.md:166 eq. 16 and PAPER.md:183 eq. 19 read
//     f_i^post = w_i  sum_{abc, a+b+c<=3}  Kt_abc  h_a(c_ix) h_b(c_iy) h_c(c_iz),
//     Kt_abc = K_abc / (norm_a norm_b norm_c),
// with the 17 Hermite coefficients
//     K_000 = rho                      (deviation form: drho, note N1)
//     K_100 = rho u_x                  (x3)
//     K_200 = rho u_x^2 + (1-omega) Pi^neq_xx,  K_110 = rho u_x u_y + (1-omega) Pi^neq_xy   (x6)
//     K_210 = a3_xxy = rho u_x^2 u_y + (1-omega)(Pi_xx u_y + 2 Pi_xy u_x)                    (x6)
//     K_111 = a3_xyz = rho u_x u_y u_z + (1-omega)(Pi_xy u_z + Pi_xz u_y + Pi_yz u_x)
// (H3_xxx == 0 on this lattice, so there is no K_300.)  The rho c_s^2 delta part of the second
// moment lives in the order-0 term (reading A17).
#pragma once
#include "tslb_common.cuh"
#include "tslb_pair.cuh"

namespace tslb {

// order of the 17 coefficients
enum KIdx {
  K000 = 0,
  K100, K010, K001,
  K200, K020, K002, K110, K101, K011,
  K210, K201, K120, K021, K102, K012, K111,
  NK
};

// Normalised post-collision coefficients Kt of one node.  V is a scalar or a small vector type
// with + and * (float, double, packed pairs).  ORDER 2 drops the third-order coefficients
// (eq. 8).
template <int ORDER, typename V>
__device__ __forceinline__ void post_collision_coeffs(V drho, V ux, V uy, V uz, V pxx, V pyy, V pzz,
                                                      V pxy, V pxz, V pyz, V omc, V *Kt) {
  const V rho = drho + V(1);
  const V mx = rho * ux, my = rho * uy, mz = rho * uz;
  const V qxx = omc * pxx, qyy = omc * pyy, qzz = omc * pzz;
  const V qxy = omc * pxy, qxz = omc * pxz, qyz = omc * pyz;
  const V axx = mx * ux + qxx, ayy = my * uy + qyy, azz = mz * uz + qzz;
  const V axy = mx * uy + qxy, axz = mx * uz + qxz, ayz = my * uz + qyz;
  Kt[K000] = drho;
  Kt[K100] = V(3) * mx;
  Kt[K010] = V(3) * my;
  Kt[K001] = V(3) * mz;
  Kt[K200] = V(4.5) * axx;
  Kt[K020] = V(4.5) * ayy;
  Kt[K002] = V(4.5) * azz;
  Kt[K110] = V(9) * axy;
  Kt[K101] = V(9) * axz;
  Kt[K011] = V(9) * ayz;
  if (ORDER >= 3) {
    const V two = V(2);
    Kt[K210] = V(13.5) * (axx * uy + two * qxy * ux);
    Kt[K201] = V(13.5) * (axx * uz + two * qxz * ux);
    Kt[K120] = V(13.5) * (ayy * ux + two * qxy * uy);
    Kt[K021] = V(13.5) * (ayy * uz + two * qyz * uy);
    Kt[K102] = V(13.5) * (azz * ux + two * qxz * uz);
    Kt[K012] = V(13.5) * (azz * uy + two * qyz * uz);
    Kt[K111] = V(27) * (axy * uz + qxz * uy + qyz * ux);
  } else {
    Kt[K210] = Kt[K201] = Kt[K120] = Kt[K021] = Kt[K102] = Kt[K012] = Kt[K111] = V(0);
  }
}

// Reading A18 (include/tslb.h TSLB_FORCING_GUO; Guo, Zheng & Shi 2002): the same coefficients for a
// node whose stored moments are the BARE ones (u_b = m/rho, Pi_b^neq relative to u_b) and which
// carries the force F.  Collision velocity u = u_b + F/(2 rho); non-equilibrium stress relative to
// u: Pi^neq = Pi_b^neq + rho (u_b u_b - u u); and on top of f^eq(u) + (1-omega) f^neq(Pi^neq, u):
//   first order   rho u + (1-omega)(m - rho u) + (1-omega/2) F  =  rho u + F/2        (= m + F)
//   second order  + (1-omega/2)(u F + F u)                          (moments of the source S_i)
// The source has no third-order part, so K_210.. K_111 are those of the unforced formula.
template <int ORDER, typename V>
__device__ __forceinline__ void post_collision_coeffs_guo(V drho, V ubx, V uby, V ubz, V pxx, V pyy, V pzz,
                                                          V pxy, V pxz, V pyz, V fx, V fy, V fz, V omc, V *Kt) {
  const V rho = drho + V(1);
  const V h = V(0.5) / rho;
  const V ux = ubx + fx * h, uy = uby + fy * h, uz = ubz + fz * h;
  post_collision_coeffs<ORDER, V>(drho, ux, uy, uz,
                                  pxx + (rho * ubx * ubx - rho * ux * ux), pyy + (rho * uby * uby - rho * uy * uy),
                                  pzz + (rho * ubz * ubz - rho * uz * uz), pxy + (rho * ubx * uby - rho * ux * uy),
                                  pxz + (rho * ubx * ubz - rho * ux * uz), pyz + (rho * uby * ubz - rho * uy * uz),
                                  omc, Kt);
  const V s = V(0.5) * (V(1) + omc);   // 1 - omega/2
  Kt[K100] += V(1.5) * fx;
  Kt[K010] += V(1.5) * fy;
  Kt[K001] += V(1.5) * fz;
  Kt[K200] += V(9) * s * (ux * fx);
  Kt[K020] += V(9) * s * (uy * fy);
  Kt[K002] += V(9) * s * (uz * fz);
  Kt[K110] += V(9) * s * (ux * fy + uy * fx);
  Kt[K101] += V(9) * s * (ux * fz + uz * fx);
  Kt[K011] += V(9) * s * (uy * fz + uz * fy);
}

// Un-normalised Hermite coefficients K_abc (same 17, same order) with explicit FMAs, for the
// tiled kernel where V is a packed pair; the 1/norm factors are folded into the 1-D operators.
template <int ORDER, typename V>
__device__ __forceinline__ void hermite_coeffs(V drho, V ux, V uy, V uz, V pxx, V pyy, V pzz, V pxy, V pxz,
                                               V pyz, V omc, V *K) {
  const V rho = drho + V(1);
  const V mx = rho * ux, my = rho * uy, mz = rho * uz;
  const V qxy = omc * pxy, qxz = omc * pxz, qyz = omc * pyz;
  const V axx = pfma(mx, ux, omc * pxx), ayy = pfma(my, uy, omc * pyy), azz = pfma(mz, uz, omc * pzz);
  const V axy = pfma(mx, uy, qxy), axz = pfma(mx, uz, qxz), ayz = pfma(my, uz, qyz);
  K[K000] = drho;
  K[K100] = mx; K[K010] = my; K[K001] = mz;
  K[K200] = axx; K[K020] = ayy; K[K002] = azz;
  K[K110] = axy; K[K101] = axz; K[K011] = ayz;
  if (ORDER >= 3) {
    const V txy = qxy + qxy, txz = qxz + qxz, tyz = qyz + qyz;
    K[K210] = pfma(txy, ux, axx * uy);
    K[K201] = pfma(txz, ux, axx * uz);
    K[K120] = pfma(txy, uy, ayy * ux);
    K[K021] = pfma(tyz, uy, ayy * uz);
    K[K102] = pfma(txz, uz, azz * ux);
    K[K012] = pfma(tyz, uz, azz * uy);
    K[K111] = pfma(qyz, ux, pfma(qxz, uy, axy * uz));
  } else {
    K[K210] = K[K201] = K[K120] = K[K021] = K[K102] = K[K012] = K[K111] = V(0);
  }
}

// 1-D basis value h_a(c) and weight w(c) for a compile-time-foldable c in {-1,0,1}
template <typename T>
__device__ __forceinline__ T h1d(int a, int c) {
  return a == 0 ? T(1) : (a == 1 ? T(c) : T(c * c) - T(1.0 / 3.0));
}
template <typename T>
__device__ __forceinline__ T w1d(int c) {
  return c == 0 ? T(2.0 / 3.0) : T(1.0 / 6.0);
}

// Finish a node: from the ten Hermite moments of the streamed populations
//   M000 = drho', M100.. = m', M200.. = Pi'_aa - rho'/3, M110.. = Pi'_ab
// to the bare velocity u_b = m'/rho' and Pi^neq' = Pi' - rho' u_b u_b - rho' c_s^2 delta
// (PAPER.md:79, 101-108).  The O(1/3) term never appears (N1).
template <typename T>
__device__ __forceinline__ void finish_moments(const T M[10], T &drho, T ub[3], T pin[6]) {
  drho = M[0];
  const T rho = T(1) + drho;
  const T inv = T(1) / rho;
  ub[0] = M[1] * inv; ub[1] = M[2] * inv; ub[2] = M[3] * inv;
  pin[0] = M[4] - M[1] * ub[0];
  pin[1] = M[5] - M[2] * ub[1];
  pin[2] = M[6] - M[3] * ub[2];
  pin[3] = M[7] - M[1] * ub[1];
  pin[4] = M[8] - M[1] * ub[2];
  pin[5] = M[9] - M[2] * ub[2];
}

}  // namespace tslb
