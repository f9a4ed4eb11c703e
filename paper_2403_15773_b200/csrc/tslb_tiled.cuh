// tslb_tiled.cuh -- the fused TSLB step as ONE TMA-staged kernel (sm_100a).
//
// Work decomposition.  A CTA owns an x-y tile of TX x TY nodes and MARCHES along z
// over a chunk of planes.  Per plane k it receives, by TMA (cp.async.bulk.tensor, one 4-D box for
// the ten moment arrays and one 3-D box for phi, completion on an mbarrier), the old moments of
// plane k on tile+halo and the old phi of plane k+1 into shared-memory rings, prefetched two planes
// ahead.  Every thread owns TWO x-adjacent nodes (packed fp32 math, tslb_pair.cuh).
//
// The 27-neighbour pull of PAPER.md:98 eq. 6 / Fig. 1 is evaluated in the tensor-product Hermite
// basis (tslb_math.cuh) as three 1-D three-point passes:
//   x-pass  (segment 1)  K_abc (17 per node, evaluated once) in push form: a+ / a- cross to the
//                        neighbouring lane inside the warp -> X^p_bc (24 per node, registers);
//   y-push  (seg. 1->2)  every row forms, per (p,c), the combination a+ it sends to the row above,
//                        a- it sends to the row below and a0 it keeps: only 9+9 values per node
//                        cross shared memory (not 24 x 3 rows) -> Y^pq_c (18, registers);
//   z-push  (segment 2)  Y^pq_c of source plane k is pushed into the register accumulators of
//                        the destination planes k-1, k, k+1 (two live accumulator sets);
// so each stored moment is read from HBM once and the populations never exist in memory.
// The phase-field half (eqs. 20-24) runs in the same kernel from the phi ring:
// y-z pre-combinations T,U,V of phi (aux warps), G and n = G/(|G|+eps) on tile+1 into a 3-plane
// ring, z-combinations of n, kappa = -div n, the kick, and the D3Q7 update assembled from
// per-plane fluxes -- phi, grad(phi), n and kappa never touch HBM.
//
// Thread roles: TY "compute" rows own the tile; 4 "aux" rows: two do the x-pass of the two halo rows,
// two the phi pre-combinations, all four the ring of the n field.  Two __syncthreads per plane.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <string>

#include "../../include/tslb.h"
#include "tslb_generic.cuh"

namespace tslb {

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *tm, uint64_t *bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, uint64_t *bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

// ------------------------------------------------------------------ configuration
template <typename T, int TX_, int TY_, bool TWO>
struct TileCfg {
  static constexpr int TX = TX_, TY = TY_;
  static constexpr int LX = TX / 2;        // threads per row (two nodes each)
  // left/right staged halo columns.  2 are needed; the TMA box row must be a multiple of 32 bytes
  // (16-byte-odd rows raised "illegal instruction" on B200), so fp32 stages 4.
  static constexpr int HL = sizeof(T) == 4 ? 4 : 2;
  static constexpr int RX = TX + 2 * HL;   // staged columns x0-HL .. x0+TX+HL-1
  static constexpr int RY = TY + 2;        // staged moment rows y0-1 .. y0+TY   ("region rows")
  static constexpr int RYP = TY + 4;       // staged phi rows y0-2 .. y0+TY+1
  static constexpr int S = 3;              // moment ring (planes k-1, k, k+1)
  static constexpr int SP = 4;             // phi ring
  static constexpr int NR = 3;             // ring of n planes
  // thread rows: TY compute rows + 4 aux rows (2 do the x-pass of the halo rows, 2 the phi
  // pre-combinations; all 4 the ring of n).  TY + 4 warps divide evenly over the 4 schedulers.
  static constexpr int NTHREADS = LX * (TY + 4);
  static constexpr int NAUX = 4 * LX;
  static constexpr int NYP = 9;            // y-push fields per direction: (p,c)
  static constexpr size_t al(size_t b) { return (b + 127) / 128 * 128; }
  static constexpr size_t MOM_BYTES = (size_t)10 * RY * RX * sizeof(T);   // one TMA box
  static constexpr size_t PHI_BYTES = (size_t)RYP * RX * sizeof(T);
  static constexpr size_t MOM_STAGE = al(MOM_BYTES);
  static constexpr size_t PHI_STAGE = al(PHI_BYTES);
  static constexpr size_t PLANE = al((size_t)RY * RX * sizeof(T));        // one region-plane array
  static constexpr size_t YP_FIELD = al((size_t)RY * TX * sizeof(T));
  static constexpr size_t OFF_MOM = 0;
  static constexpr size_t OFF_PHI = OFF_MOM + S * MOM_STAGE;
  static constexpr size_t OFF_TUV = OFF_PHI + (TWO ? SP * PHI_STAGE : 0);  // T, U, V of plane k
  static constexpr size_t OFF_NRM = OFF_TUV + (TWO ? 3 * PLANE : 0);       // n ring [NR][3]
  static constexpr size_t OFF_ZC = OFF_NRM + (TWO ? NR * 3 * PLANE : 0);   // S_z n_x, S_z n_y, d_z n_z
  static constexpr size_t OFF_AP = OFF_ZC + (TWO ? 3 * PLANE : 0);         // y-push, upward  [9]
  static constexpr size_t OFF_AM = OFF_AP + NYP * YP_FIELD;                // y-push, downward [9]
  // x exchange.  Inside a warp the a+ of each pair's second node / a- of its first node cross
  // through the warp's OWN first row of the y-push fields 0..7 (dead at that time).  Only the terms
  // of the two halo columns x0-1 (a+) and x0+TX (a-) need storage of their own: [2][8][RY].
  static constexpr size_t XH_BYTES = al((size_t)2 * 8 * RY * sizeof(T));
  static constexpr size_t OFF_XH = OFF_AM + NYP * YP_FIELD;
  static constexpr size_t OFF_BAR = OFF_XH + XH_BYTES;
  static constexpr size_t SMEM_BYTES = OFF_BAR + 64;
};

struct TiledMaps {
  CUtensorMap mom;   // 4-D (px, py, nz, 10) over the SOURCE buffer, box (RX, RY, 1, 10)
  CUtensorMap phi;   // 3-D (px, py, nz) over the source phi, box (RX, RYP, 1)
  int ntx, nty;      // tiles per row / column
  int zc;            // planes per z chunk
};

// Reciprocal and square root.  fp32: the branch-free MUFU approximations (<= 2 ulp, far inside the
// 1e-5 parity gate; rho' ~ 1 and |G| + eps >= 1e-12 are normal numbers); fp64: IEEE.
__device__ __forceinline__ float rcp1(float s) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s)); return r; }
__device__ __forceinline__ double rcp1(double s) { return 1.0 / s; }
__device__ __forceinline__ float sqrt1(float s) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s)); return r; }
__device__ __forceinline__ double sqrt1(double s) { return sqrt(s); }
template <typename T> __device__ __forceinline__ Pair<T> prcp(Pair<T> a) { return Pair<T>(rcp1(a.x), rcp1(a.y)); }

// The 1-D three-point operator of the tensor-product basis in PUSH form.  A source
// node holding the un-normalised Hermite coefficients g_0, g_1, g_2 (index along this axis) sends
//     a+ = g0/6 + g1/2 + g2/2   to the node at +1,
//     a- = g0/6 - g1/2 + g2/2   to the node at -1,  and keeps  a0 = 2 g0/3 - g2;
// the destination's Hermite moments along the axis are then
//     W0 = a+(-1) + a0 + a-(+1),   W1 = a+(-1) - a-(+1),   W2 = 2/3 (a+(-1) + a-(+1)) - a0/3.
// (w(+-1) = 1/6, w(0) = 2/3, norms 1, 1/3, 2/9: a+ = w h_a(+1)/norm_a summed over a, etc.)
template <int NA, typename V, typename T>
__device__ __forceinline__ void push3(V g0, V g1, V g2, V &ap, V &am, V &a0) {
  V h = g0 * T(1.0 / 6.0);
  if (NA == 3) h = pfma(g2, T(0.5), h);
  ap = h; am = h;
  if (NA >= 2) { ap = pfma(g1, T(0.5), h); am = pfma(g1, T(-0.5), h); }
  a0 = NA == 3 ? pfma(g0, T(2.0 / 3.0), pneg(g2)) : g0 * T(2.0 / 3.0);
}
// destination side: from up = a+(-1), dn = a-(+1), a0 -> W0, W1, W2
template <typename V, typename T>
__device__ __forceinline__ void pull3(V up, V dn, V a0, V &W0, V &W1, V &W2) {
  const V s = up + dn;
  W0 = s + a0;
  W1 = up - dn;
  W2 = pfma(W0, T(2.0 / 3.0), pneg(a0));     // = 2/3 s - a0/3
}
// the same with up = (l, upy) and dn = (dnx, r) given as scalars from two different register pairs
template <typename V, typename T>
__device__ __forceinline__ void pull3s(T l, T upy, T dnx, T r, V a0, V &W0, V &W1, V &W2) {
  const V s(l + dnx, upy + r);
  W0 = s + a0;
  W1 = V(l - dnx, upy - r);
  W2 = pfma(W0, T(2.0 / 3.0), pneg(a0));
}

// ------------------------------------------------------------------ the kernel
// SLAB: the context is a z-slab (halo faces, ghost planes, halo push).  A separate instantiation:
// the single-GPU kernel's loop body sits at the 32 KB instruction-cache limit and must not grow.
template <typename T, int TX, int TY, int ORDER, bool TWO, bool SLAB>
__global__ void __launch_bounds__((TX / 2) * (TY + 4), (TileCfg<T, TX, TY, TWO>::SMEM_BYTES <= 113 * 1024 ? 2 : 1))
tiled_step_kernel(const __grid_constant__ StepParams<T> P, const __grid_constant__ TiledMaps M) {
  using C = TileCfg<T, TX, TY, TWO>;
  using V = Pair<T>;
  constexpr int LX = C::LX, HL = C::HL, RX = C::RX, RY = C::RY, S = C::S, SP = C::SP, NR = C::NR;
  constexpr int PL = (int)(C::PLANE / sizeof(T));       // elements per region-plane array
  constexpr int YPF = (int)(C::YP_FIELD / sizeof(T));   // elements per y-push field
  constexpr int MF = RY * RX;                           // elements per moment field in a stage
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::OFF_BAR);
  auto mom_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_MOM + slot * C::MOM_STAGE); };
  auto phi_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_PHI + slot * C::PHI_STAGE); };
  auto nrm_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_NRM + slot * 3 * C::PLANE); };
  T *s_tuv = reinterpret_cast<T *>(smem + C::OFF_TUV);
  T *s_zc = reinterpret_cast<T *>(smem + C::OFF_ZC);
  T *s_ap = reinterpret_cast<T *>(smem + C::OFF_AP);
  T *s_am = reinterpret_cast<T *>(smem + C::OFF_AM);
  T *s_xhl = reinterpret_cast<T *>(smem + C::OFF_XH);      // a+ of column x0-1   [8][RY]
  T *s_xhr = s_xhl + 8 * RY;                                // a- of column x0+TX  [8][RY]

  const Layout &L = P.L;
  const int t = threadIdx.x;
  const int lx = t % LX;
  const int tr = t / LX;
  const bool aux = tr >= TY;
  const bool xrow = tr < TY + 2;                          // does an x-pass row
  const int r = aux ? (tr == TY ? 0 : RY - 1) : tr + 1;   // region row (y = y0 - 1 + r)
  const int c0 = HL + 2 * lx;                             // staged column of the pair's first node
  const int oM = r * RX + c0;                             // offset of the pair in a region plane
  const int oY = r * TX + 2 * lx;                         // offset of the pair in a y-push field
  // region-plane offset of the ring column next to the pair for the lanes at the tile edge; one
  // common (valid) word for all other lanes
  const int eoff = lx == 0 ? oM - 1 : (lx == LX - 1 ? oM + 2 : RX + HL);
  const int ia = (tr - TY) * LX + lx;                     // aux thread index
  // x-exchange word of this lane: word (t & 31) of the y-push row owned by lane 0 of the warp
  const int trf = (t & ~31) / LX;
  const int oX = (trf < TY ? trf + 1 : (trf == TY ? 0 : RY - 1)) * TX + (t & 31);
  // Tile origin.  When nx (ny) is not a multiple of the tile, the last tile of the row (column) is
  // shifted back to end at the domain edge; it recomputes the overlap but stores only its own nodes.
  const int xs = (blockIdx.x % M.ntx) * TX, ys = (blockIdx.x / M.ntx) * TY;
  const int x0 = min(xs, L.nx - TX), y0 = min(ys, L.ny - TY);
  const int z0 = blockIdx.y * M.zc;
  const int z1 = min(z0 + M.zc, L.nz);
  const int kb = z0 - 1;                 // first source plane
  const int NG = z1 - kb + 1;            // load groups / x-pass planes: kb .. z1
  const int NI = NG + 1;                 // iterations

  // plane coordinate in the tensor map: wrapped / clamped / ghost plane of a slab (zsrc), shifted
  // by the ghost planes below z = 0
  auto zmap = [&](int z) { return zsrc(P, z) + L.gz; };
  // group g (relative index): moments of plane kb+g -> slot g%S, phi of plane kb+g+1 -> slot (g+2)%SP
  auto issue = [&](int g) {
    uint64_t *bar = &bars[g % S];
    uint32_t bytes = (uint32_t)C::MOM_BYTES + (TWO ? (uint32_t)C::PHI_BYTES : 0u);
    if (TWO && g == 0) bytes += 2u * (uint32_t)C::PHI_BYTES;
    mbar_expect_tx(bar, bytes);
    tma_load_4d(mom_at(g % S), &M.mom, bar, x0 - HL + GX, y0 - 1 + GY, zmap(kb + g), 0);
    if (TWO) {
      tma_load_3d(phi_at((g + 2) % SP), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb + g + 1));
      if (g == 0) {
        tma_load_3d(phi_at(0), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb - 1));
        tma_load_3d(phi_at(1), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb));
      }
    }
  };

  if (t == 0) {
    for (int s = 0; s < S; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  const V omc(P.omc);
  const T w1 = T(1.0 / 6.0), w0 = T(2.0 / 3.0);
  V accA[10], accB[10];     // Hermite moments being accumulated for planes k and k+1
  V fl[10];                 // finished flow part of the plane completed in the previous iteration:
                            // drho', u_b (3), Pi^neq' (6)
  V A0[9];                  // this row's own y-push term a0 per (c,p), carried across the barrier
  V nA[3], nB[3];           // own n of planes k-2 and k-1
  V gA(T(0)), gB(T(0));     // own |G| of planes k-2 and k-1
  V c_inpl(T(0)), c_upa(T(0)), c_upb(T(0)), c_rinv(T(1));
#pragma unroll
  for (int m = 0; m < 10; ++m) { accA[m] = V(T(0)); accB[m] = V(T(0)); fl[m] = V(T(0)); }
#pragma unroll
  for (int m = 0; m < 3; ++m) { nA[m] = V(T(0)); nB[m] = V(T(0)); }

  // global store offsets of the pair (plane 0); the periodic ghost images of edge nodes
  const int gx_ = x0 + 2 * lx, gy_ = y0 + tr;
  const int gxg = gx_ < 2 ? gx_ + L.nx : (gx_ >= L.nx - 2 ? gx_ - L.nx : gx_);
  const int gyg = gy_ < GY ? gy_ + L.ny : (gy_ >= L.ny - GY ? gy_ - L.ny : gy_);
  const bool own = gx_ >= xs && gy_ >= ys;
  const long long o00 = L.idx(gx_, gy_, 0), o10 = L.idx(gxg, gy_, 0), o01 = L.idx(gx_, gyg, 0), o11 = L.idx(gxg, gyg, 0);

  // x-pass terms of the two halo columns x0-1 (its a+) and x0+TX (its a-) of every region row of
  // the plane held in moment slot `slot`; done by the A1 aux threads one segment ahead.
  auto halo_cols = [&](int slot) {
    const int e = ia - 2 * LX;
    if (e >= 0 && e < 2 * RY) {
      const int rr = e >> 1, side = e & 1;
      const T *p = mom_at(slot) + rr * RX + (side ? HL + TX : HL - 1);
      T m[10], K[NK];
#pragma unroll
      for (int f = 0; f < 10; ++f) m[f] = p[f * MF];
      hermite_coeffs<ORDER, T>(m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], m[8], m[9], P.omc, K);
      T gp[8], gm[8], g0;
      push3<3, T, T>(K[K000], K[K100], K[K200], gp[0], gm[0], g0);
      push3<3, T, T>(K[K010], K[K110], K[K210], gp[1], gm[1], g0);
      push3<2, T, T>(K[K020], K[K120], K[K120], gp[2], gm[2], g0);
      push3<3, T, T>(K[K001], K[K101], K[K201], gp[3], gm[3], g0);
      push3<2, T, T>(K[K011], K[K111], K[K111], gp[4], gm[4], g0);
      push3<1, T, T>(K[K021], K[K021], K[K021], gp[5], gm[5], g0);
      push3<2, T, T>(K[K002], K[K102], K[K102], gp[6], gm[6], g0);
      push3<1, T, T>(K[K012], K[K012], K[K012], gp[7], gm[7], g0);
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        if (side == 0) s_xhl[g * RY + rr] = gp[g];
        else s_xhr[g * RY + rr] = gm[g];
      }
    }
  };
  // Ring slots of iteration i: moments i%S, phi(k-1) i%SP, n(k) i%NR.  Iterations -2 and -1 are the
  // pipeline prologue run through the same code (first two TMA groups, halo columns of the first
  // plane): one copy of issue() and halo_cols() keeps the loop inside the instruction cache.
  int ms = S - 2, ps = SP - 2, ns = NR - 2;
  uint32_t mph = 1;                      // mbarrier phase parity of slot ms (flips when ms wraps to 0)
  for (int i = -2; i < NI; ++i) {
    const int k = kb + i;
    const bool act = (unsigned)i < (unsigned)NG;       // plane k is a source plane of this chunk
    if (act) mbar_wait(&bars[ms], mph);
    const int ms1 = ms == 0 ? S - 1 : ms - 1;          // moments of plane k-1
    const int ns1 = ns == 0 ? NR - 1 : ns - 1;         // n of plane k-1
    const int ns2 = ns1 == 0 ? NR - 1 : ns1 - 1;       // n of plane k-2
    const T *phm = phi_at(ps);                         // phi(k-1)
    const T *phc = phi_at((ps + 1) % SP);              // phi(k)
    const T *php = phi_at((ps + 2) % SP);              // phi(k+1)

    // =========================== segment 1 ===========================
    if (TWO && !xrow && act) {
      // A1: T = S_y S_z phi, U = d_y S_z phi, V = S_y d_z phi of plane k on the region rows
      // one thread per column pair, marching down the rows with a 3-row window of S_z phi, d_z phi
      const int a1 = ia - 2 * LX;
      if (a1 < RX / 2) {
        const int cp = 2 * a1;
        V sz0, sz1, sz2, dz0, dz1, dz2;
        auto zrow = [&](int prow, V &sz, V &dz) {
          const V a = lds_pair(phm + prow * RX + cp), b = lds_pair(phc + prow * RX + cp), c = lds_pair(php + prow * RX + cp);
          sz = pfma(b, w0, (a + c) * w1);
          dz = (c - a) * T(0.5);
        };
        zrow(0, sz0, dz0);
        zrow(1, sz1, dz1);
#pragma unroll
        for (int rr = 0; rr < RY; ++rr) {
          zrow(rr + 2, sz2, dz2);
          sts_pair(s_tuv + rr * RX + cp, pfma(sz1, w0, (sz0 + sz2) * w1));
          sts_pair(s_tuv + PL + rr * RX + cp, (sz2 - sz0) * T(0.5));
          sts_pair(s_tuv + 2 * PL + rr * RX + cp, pfma(dz1, w0, (dz0 + dz2) * w1));
          sz0 = sz1; sz1 = sz2; dz0 = dz1; dz1 = dz2;
        }
      }
    }
    if (!aux && i >= 1) {
      V phin(T(0)), ukx(T(0)), uky(T(0)), ukz(T(0));
      const int j = k - 2;                         // plane finalised in this iteration
      const bool fin = (j >= z0);                  // (j < z1 always: k <= z1 + 1)
      if (TWO) {
        // fluxes of plane k-1 (operands resident: moments slot ms1, phi(k-1) = phm, n(k-1) slot ns1)
        const T *ph = phm + (r + 1) * RX + c0;
        const T *mo = mom_at(ms1) + oM;
        const T *nr = nrm_at(ns1) + oM;
        // q = phi (4 c.u + gamma (1-phi) c.n): the neighbour sends phi + q along +e, phi - q along -e
        const V gamv(P.gamma);
        auto qterm = [&](V p, V u, V n) { return p * pfma(pfma(p, V(T(0)) - gamv, gamv), n, u * T(4)); };
        const V pc = lds_pair(ph);
        // x direction: node x gets g+(c0-1) + g-(c0+1), node x+1 gets g+(c0) + g-(c0+2)
        const V uxc = lds_pair(mo + F_UX * MF);
        // (q on the own columns and on the two outer columns c0-1, c0+2; mixed only at the end)
        const V pn(ph[-1], ph[2]);
        const V qO = qterm(pc, uxc, nB[0]);
        const V qX = qterm(pn, V(mo[F_UX * MF - 1], mo[F_UX * MF + 2]), V(nr[-1], nr[2]));
        V inpl((pn.x + qX.x) + (pc.y - qO.y), (pc.x + qO.x) + (pn.y - qX.y));
        // y direction: rows r-1 (south, c_i = +e_y) and r+1 (north)
        const V phs = lds_pair(ph - RX), phn_ = lds_pair(ph + RX);
        const V qS = qterm(phs, lds_pair(mo + F_UY * MF - RX), lds_pair(nr + PL - RX));
        const V qN = qterm(phn_, lds_pair(mo + F_UY * MF + RX), lds_pair(nr + PL + RX));
        inpl = inpl + ((phs + qS) + (phn_ - qN));
        inpl = pfma(inpl, T(0.125), pc * T(0.25));
        // z direction: this plane's contribution to the planes above (up) and below (down)
        const V qZ = qterm(pc, lds_pair(mo + F_UZ * MF), nB[2]);
        const V up = pc + qZ, down = pc - qZ;
        if (fin) {
          // a7: phi'(j) = inpl(j) + up(j-1)/8 + down(j+1)/8       (eqs. 23-24)
          phin = pfma(c_upa + down, T(0.125), c_inpl);
          // a5: kappa(j) = -div n from the z-combined normals a = S_z n_x, b = S_z n_y, c = d_z n_z
          // Own columns from shared memory; the outer columns c0-1 / c0+2 come from the neighbour
          // lanes by shuffle (3x the LSU rate, no bank conflicts).  The lanes at the tile edge read
          // the ring column instead: one unconditional load per term through a per-lane pointer
          // (all other lanes read one common word: a broadcast), no divergence.
          const T *za = s_zc + oM, *zb = za + PL, *zc_ = za + 2 * PL;
          V own(T(0)), eO(T(0));
#pragma unroll
          for (int dy = -1; dy <= 1; ++dy) {
            const T w = dy == 0 ? w0 : w1;
            own = pfma(lds_pair(za + dy * RX), w, own);       // S_y a
            eO = pfma(lds_pair(zc_ + dy * RX), w, eO);         // S_y c
          }
          const V dO = lds_pair(zb + RX) - lds_pair(zb - RX);  // 2 d_y b
          const T *ze = s_zc + eoff;                           // ring column (edge lanes) / dummy
          const T ea = w1 * (ze[-RX] + ze[RX]) + w0 * ze[0];
          const T ec = w1 * (ze[2 * PL - RX] + ze[2 * PL + RX]) + w0 * ze[2 * PL];
          const T eb = ze[PL + RX] - ze[PL - RX];
          auto left = [&](T v, T e) { const T q = __shfl_up_sync(0xffffffffu, v, 1, LX); return lx == 0 ? e : q; };
          auto right = [&](T v, T e) { const T q = __shfl_down_sync(0xffffffffu, v, 1, LX); return lx == LX - 1 ? e : q; };
          const T al = left(own.y, ea), ar = right(own.x, ea);
          const T bl = left(dO.y, eb), br = right(dO.x, eb);
          const T cl = left(eO.y, ec), cr = right(eO.x, ec);
          V kap(T(0.5) * (own.y - al), T(0.5) * (ar - own.x));                     // d/dx S_y a
          kap.x += T(0.5) * (w1 * bl + w0 * dO.x + w1 * dO.y);                       // S_x d/dy b
          kap.y += T(0.5) * (w1 * dO.x + w0 * dO.y + w1 * br);
          kap.x += w1 * cl + w0 * eO.x + w1 * eO.y;                                  // S_x S_y c
          kap.y += w1 * eO.x + w0 * eO.y + w1 * cr;
          // a6: F = sigma kappa G, kappa = -div n, G = n (|G| + eps); u' = u_b + F / rho'
          const V sc = (kap * (gA + V(T(1e-12)))) * c_rinv * (-P.sigma);
          ukx = nA[0] * sc; uky = nA[1] * sc; ukz = nA[2] * sc;
        }
        c_upa = c_upb; c_upb = up; c_inpl = inpl;
      }
      if (fin && own && !((P.jet_lo && j == 0) || (P.out_hi && j == L.nz - 1))) {
        // a9: store plane j (and its periodic ghost images)
        V o[NF_MAX];
        o[0] = fl[0];
        o[1] = fl[1] + ukx; o[2] = fl[2] + uky; o[3] = fl[3] + ukz;
#pragma unroll
        for (int m = 4; m < 10; ++m) o[m] = fl[m];
        o[10] = phin;
        const long long zo = (long long)j * L.plane;
#pragma unroll
        for (int m = 0; m < (TWO ? 11 : 10); ++m) *reinterpret_cast<V *>(P.out.f[m] + zo + o00) = o[m];
        if (gxg != gx_ || gyg != gy_) {          // periodic ghost images (edge tiles only)
#pragma unroll 1
          for (int im = 0; im < 3; ++im) {       // one copy of the store code: x image, y image, corner
            if (im == 0 ? gxg == gx_ : (im == 1 ? gyg == gy_ : (gxg == gx_ || gyg == gy_))) continue;
            const long long og = zo + (im == 0 ? o10 : (im == 1 ? o01 : o11));
#pragma unroll
            for (int m = 0; m < (TWO ? 11 : 10); ++m) *reinterpret_cast<V *>(P.out.f[m] + og) = o[m];
          }
        }
        // halo push (slab faces only, off the common path): the same stores into the neighbour
        // slab's ghost planes through its peer pointers -- phi from the two planes next to the
        // face, the moments from the face plane
        if (SLAB && ((j < 2 && P.nb[0].f[0]) || (j >= L.nz - 2 && P.nb[1].f[0]))) {
#pragma unroll 1
          for (int side = 0; side < 2; ++side) {
            const int depth = side == 0 ? j : L.nz - 1 - j;
            if (!P.nb[side].f[0] || depth > 1) continue;
            const long long zn = (long long)(j + P.nb_dz[side]) * L.plane;
#pragma unroll 1
            for (int im = 0; im < 4; ++im) {     // the node itself, then its x / y / corner images
              if (im == 1 ? gxg == gx_ : (im == 2 ? gyg == gy_ : (im == 3 && (gxg == gx_ || gyg == gy_)))) continue;
              const long long og = zn + (im == 0 ? o00 : (im == 1 ? o10 : (im == 2 ? o01 : o11)));
#pragma unroll
              for (int m = 0; m < (TWO ? 11 : 10); ++m)
                if (depth == 0 || m == F_PHI) *reinterpret_cast<V *>(P.nb[side].f[m] + og) = o[m];
            }
          }
        }
      }
    }
    if (xrow && act) {
      // A2: x-pass of region row r of plane k in push form, then the y-push terms.  Each node's K is
      // evaluated once; a+ / a- cross to the x-neighbour thread through shared memory (same warp).
      V Xg[8][3];   // [group][p]
      {
        V m[10], K[NK];
        const T *p = mom_at(ms) + oM;
#pragma unroll
        for (int f = 0; f < 10; ++f) m[f] = lds_pair(p + f * MF);
        hermite_coeffs<ORDER, V>(m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], m[8], m[9], omc, K);
        V gp[8], gm[8], g0[8];
        push3<3, V, T>(K[K000], K[K100], K[K200], gp[0], gm[0], g0[0]);   // (b,c) = (0,0)
        push3<3, V, T>(K[K010], K[K110], K[K210], gp[1], gm[1], g0[1]);   // (1,0)
        push3<2, V, T>(K[K020], K[K120], K[K120], gp[2], gm[2], g0[2]);   // (2,0)
        push3<3, V, T>(K[K001], K[K101], K[K201], gp[3], gm[3], g0[3]);   // (0,1)
        push3<2, V, T>(K[K011], K[K111], K[K111], gp[4], gm[4], g0[4]);   // (1,1)
        push3<1, V, T>(K[K021], K[K021], K[K021], gp[5], gm[5], g0[5]);   // (2,1)
        push3<2, V, T>(K[K002], K[K102], K[K102], gp[6], gm[6], g0[6]);   // (0,2)
        push3<1, V, T>(K[K012], K[K012], K[K012], gp[7], gm[7], g0[7]);   // (1,2)
        // lane l of the warp parks gp.y / gm.x at word l of the warp's first y-push row
        T *xp = s_ap + oX, *xm = s_am + oX;
#pragma unroll
        for (int g = 0; g < 8; ++g) { xp[g * YPF] = gp[g].y; xm[g * YPF] = gm[g].x; }
        __syncwarp();
        // left / right neighbour's word, or the halo column's term for the lanes at the tile edge
        const T *pl = lx == 0 ? s_xhl + r : xp - 1, *pr = lx == LX - 1 ? s_xhr + r : xm + 1;
        const int sl = lx == 0 ? RY : YPF, sr = lx == LX - 1 ? RY : YPF;
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          pull3s<V, T>(pl[g * sl], gp[g].x, gm[g].y, pr[g * sr], g0[g], Xg[g][0], Xg[g][1], Xg[g][2]);
        }
        __syncwarp();
      }
      // y-push per (c, p): groups of c = 0: b = 0,1,2 -> g 0,1,2; c = 1: g 3,4,5; c = 2: b = 0,1 -> g 6,7
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int p = 0; p < 3; ++p) {
          V ap, am;
          if (c < 2) push3<3, V, T>(Xg[3 * c][p], Xg[3 * c + 1][p], Xg[3 * c + 2][p], ap, am, A0[3 * c + p]);
          else push3<2, V, T>(Xg[6][p], Xg[7][p], Xg[7][p], ap, am, A0[6 + p]);
          sts_pair(s_ap + (3 * c + p) * YPF + oY, ap);
          sts_pair(s_am + (3 * c + p) * YPF + oY, am);
        }
    }
    __syncthreads();
    if (t == 0 && i + 2 < NG) issue(i + 2);

    // =========================== segment 2 ===========================
    if (!xrow && (unsigned)(i + 1) < (unsigned)NG) {
      const int sl = ms == S - 1 ? 0 : ms + 1;
      mbar_wait(&bars[sl], sl == 0 ? mph ^ 1u : mph);
      halo_cols(sl);
    }
    if (act) {
      if (!aux) {
        // B2: finish the y-pass (a+ from the row below, a- from the row above, own a0) and z-push.
        V outm[10];
        // moment index of (p,q,rr)
        constexpr int MI[3][3][3] = {{{0, 3, 6}, {2, 9, -1}, {5, -1, -1}}, {{1, 8, -1}, {7, -1, -1}, {-1, -1, -1}}, {{4, -1, -1}, {-1, -1, -1}, {-1, -1, -1}}};
#pragma unroll
        for (int p = 0; p < 3; ++p) {
          V Yq[3][3];   // [q][c]
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            const V up = lds_pair(s_ap + (3 * c + p) * YPF + oY - TX);
            const V dn = lds_pair(s_am + (3 * c + p) * YPF + oY + TX);
            pull3<V, T>(up, dn, A0[3 * c + p], Yq[0][c], Yq[1][c], Yq[2][c]);
          }
#pragma unroll
          for (int q = 0; q + p <= 2; ++q) {
            V ap, am, a0;
            push3<3, V, T>(Yq[q][0], Yq[q][1], Yq[q][2], ap, am, a0);   // ap -> plane k+1, am -> plane k-1
            {
              const int m = MI[p][q][0];
              outm[m] = accA[m] + am; accA[m] = accB[m] + a0; accB[m] = ap;
            }
            if (p + q <= 1) {
              const int m = MI[p][q][1];
              outm[m] = accA[m] - am; accA[m] = accB[m]; accB[m] = ap;
            }
            if (p + q == 0) {
              const int m = MI[p][q][2];
              outm[m] = pfma(am, T(2.0 / 3.0), accA[m]);
              accA[m] = pfma(a0, T(-1.0 / 3.0), accB[m]);
              accB[m] = ap * T(2.0 / 3.0);
            }
          }
        }
        // a4: plane k-1 is complete: u_b = m'/rho', Pi^neq' = Pi' - rho' u_b u_b (Hermite form)
        const V inv = prcp<T>(outm[0] + V(T(1)));
        c_rinv = inv;
        fl[0] = outm[0];
        fl[1] = outm[1] * inv; fl[2] = outm[2] * inv; fl[3] = outm[3] * inv;
        fl[4] = outm[4] - outm[1] * fl[1];
        fl[5] = outm[5] - outm[2] * fl[2];
        fl[6] = outm[6] - outm[3] * fl[3];
        fl[7] = outm[7] - outm[1] * fl[2];
        fl[8] = outm[8] - outm[1] * fl[3];
        fl[9] = outm[9] - outm[2] * fl[3];
      }
      if (TWO) {
        // B1: G = (d_x T, S_x U, S_x V), n = G/(|G|+eps) of plane k on tile+1 -> ring slot ns
        T *nk = nrm_at(ns);
        auto gn_pair = [&](int o, int ol, int orr, V nn[3], V &mag) {
          const V tc = lds_pair(s_tuv + o), uc = lds_pair(s_tuv + PL + o), vc = lds_pair(s_tuv + 2 * PL + o);
          const T tl = s_tuv[ol], tr_ = s_tuv[orr], ul = s_tuv[PL + ol], ur = s_tuv[PL + orr];
          const T vl = s_tuv[2 * PL + ol], vr = s_tuv[2 * PL + orr];
          const V gx(T(0.5) * (tc.y - tl), T(0.5) * (tr_ - tc.x));
          const V gy(w1 * (ul + uc.y) + w0 * uc.x, w1 * (uc.x + ur) + w0 * uc.y);
          const V gz(w1 * (vl + vc.y) + w0 * vc.x, w1 * (vc.x + vr) + w0 * vc.y);
          const V s2 = pfma(gz, gz, pfma(gy, gy, gx * gx));
          mag = V(sqrt1(s2.x), sqrt1(s2.y));                                  // |G|
          const V inv(rcp1(mag.x + T(1e-12)), rcp1(mag.y + T(1e-12)));             // reading A7
          nn[0] = gx * inv; nn[1] = gy * inv; nn[2] = gz * inv;
          sts_pair(nk + o, nn[0]); sts_pair(nk + PL + o, nn[1]); sts_pair(nk + 2 * PL + o, nn[2]);
        };
        if (!aux) {
          V nC[3], gC;
          gn_pair(oM, oM - 1, oM + 2, nC, gC);
          // z-combinations of the own normals for kappa(k-1)
          sts_pair(s_zc + oM, pfma(nB[0], w0, (nA[0] + nC[0]) * w1));
          sts_pair(s_zc + PL + oM, pfma(nB[1], w0, (nA[1] + nC[1]) * w1));
          sts_pair(s_zc + 2 * PL + oM, (nC[2] - nA[2]) * T(0.5));
#pragma unroll
          for (int a = 0; a < 3; ++a) { nA[a] = nB[a]; nB[a] = nC[a]; }
          gA = gB; gB = gC;
        } else {
          constexpr int PPR = TX / 2 + 2;                // pairs per full ring row: cols HL-2 .. HL+TX+1
          constexpr int NT = 2 * PPR + 2 * TY;           // ring tasks
          const T *n1 = nrm_at(ns1), *n2 = nrm_at(ns2);
          for (int e = ia; e < NT; e += C::NAUX) {
            int rr, c;
            if (e < 2 * PPR) { rr = (e < PPR) ? 0 : RY - 1; c = HL - 2 + 2 * (e % PPR); }
            else { const int q = e - 2 * PPR; rr = 1 + (q >> 1); c = (q & 1) ? HL + TX : HL - 2; }
            const int o = rr * RX + c;
            const int ol = c > 0 ? o - 1 : o, orr = c + 2 < RX ? o + 2 : o + 1;   // clamped; edge results unused
            V nC[3], gC;
            gn_pair(o, ol, orr, nC, gC);
            const V a2 = lds_pair(n2 + o), a1 = lds_pair(n1 + o);
            const V b2 = lds_pair(n2 + PL + o), b1 = lds_pair(n1 + PL + o);
            const V c2 = lds_pair(n2 + 2 * PL + o);
            sts_pair(s_zc + o, pfma(a1, w0, (a2 + nC[0]) * w1));
            sts_pair(s_zc + PL + o, pfma(b1, w0, (b2 + nC[1]) * w1));
            sts_pair(s_zc + 2 * PL + o, (nC[2] - c2) * T(0.5));
          }
        }
      }
    }
    __syncthreads();
    ms = ms == S - 1 ? 0 : ms + 1;
    if (ms == 0) mph ^= 1u;
    ps = ps == SP - 1 ? 0 : ps + 1;
    ns = ns == NR - 1 ? 0 : ns + 1;
  }
}

// ------------------------------------------------------------------ host side
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TiledPlan {
  std::string name;
  int precision = 0, tx = 0, ty = 0, zc = 0;
  TiledMaps maps[2];     // per source buffer
  bool two = false;
};

// tile shapes: 32x8 in both precisions (fp32: ~103 KB of shared memory -> two CTAs per SM, whose
// barrier phases interleave; measured 30.2 vs 27.6 GLUPS for 64x8 on C5)
#ifndef TSLB_F32_TX
#define TSLB_F32_TX 32
#endif
#ifndef TSLB_F64_TX
#define TSLB_F64_TX 32
#endif
#ifndef TSLB_TY
#define TSLB_TY 8
#endif
inline void tiled_tile(int precision, int &tx, int &ty) {
  tx = precision == TSLB_F32 ? TSLB_F32_TX : TSLB_F64_TX;
  ty = TSLB_TY;
}

inline bool tiled_supported(int precision, int nx, int ny, int nz) {
  int tx, ty;
  tiled_tile(precision, tx, ty);
  // rows of the padded arrays must be multiples of 16 bytes for TMA (px = nx + 16)
  return nx % (precision == TSLB_F32 ? 4 : 2) == 0 && nz >= 1 && nx >= tx && ny >= ty;
}

inline bool tiled_plan_create(TiledPlan &pl, int precision, const Layout &L, void *fields[2][NF_MAX], int nfields,
                              int device, std::string &why) {
  (void)device;
  PFN_encodeTiled enc = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void **)&enc, cudaEnableDefault, &qres);
  if (e != cudaSuccess || !enc || qres != cudaDriverEntryPointSuccess) {
    why = "cuTensorMapEncodeTiled not available from the driver";
    return false;
  }
  pl.precision = precision;
  pl.two = nfields == 11;
  tiled_tile(precision, pl.tx, pl.ty);
  const size_t es = precision == TSLB_F32 ? 4 : 8;
  const CUtensorMapDataType dt = precision == TSLB_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  const int RX = pl.tx + 2 * (es == 4 ? 4 : 2), RY = pl.ty + 2, RYP = pl.ty + 4;
  for (int b = 0; b < 2; ++b) {
    const size_t fstride = (size_t)((char *)fields[b][1] - (char *)fields[b][0]);
    cuuint64_t gdim[4] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)(L.nz + 2 * L.gz), 10};
    const size_t zoff = (size_t)L.gz * (size_t)L.plane * es;     // fields[][] point at plane 0
    cuuint64_t gstr[3] = {(cuuint64_t)L.px * es, (cuuint64_t)L.plane * es, (cuuint64_t)fstride};
    cuuint32_t box[4] = {(cuuint32_t)RX, (cuuint32_t)RY, 1, 10};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(&pl.maps[b].mom, dt, 4, (char *)fields[b][0] - zoff, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled(moments) failed: " + std::to_string((int)r); return false; }
    if (pl.two) {
      cuuint32_t boxp[3] = {(cuuint32_t)RX, (cuuint32_t)RYP, 1};
      r = enc(&pl.maps[b].phi, dt, 3, (char *)fields[b][F_PHI] - zoff, gdim, gstr, boxp, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled(phi) failed: " + std::to_string((int)r); return false; }
    } else {
      pl.maps[b].phi = pl.maps[b].mom;
    }
    pl.maps[b].ntx = (L.nx + pl.tx - 1) / pl.tx;
    pl.maps[b].nty = (L.ny + pl.ty - 1) / pl.ty;
  }
  // z chunking: every chunk pays a 3-plane pipeline prologue, and the grid runs in waves of
  // (CTAs per SM) x (SM count): pick the chunk length that minimises waves x (zc + 3).
  const long long tiles = (long long)pl.maps[0].ntx * pl.maps[0].nty;
  int nsm = 148;
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, device);
  const long long slots = (long long)nsm * (precision == TSLB_F32 ? 2 : 1);
  int zc = L.nz;
  long long best = -1;
  for (int cand = 8; cand <= 128; cand *= 2) {
    const int c = cand < L.nz ? cand : L.nz;
    const long long ctas = tiles * ((L.nz + c - 1) / c);
    const long long cost = ((ctas + slots - 1) / slots) * (c + 3);
    if (best < 0 || cost < best) { best = cost; zc = c; }
  }
  if (const char *env = getenv("TSLB_ZCHUNK")) { int v = atoi(env); if (v > 0) zc = v; }
  pl.zc = zc;
  pl.maps[0].zc = pl.maps[1].zc = zc;
  pl.name = "tiled<" + std::to_string(pl.tx) + "x" + std::to_string(pl.ty) + ",zc=" + std::to_string(zc) + ">";
  return true;
}

inline void tiled_plan_destroy(TiledPlan &) {}

// jet boundary planes (O9) after the tiled kernel: reads only OLD fields, writes only the two
// boundary planes of the NEW buffer (+ their ghosts)
template <typename T>
__global__ void tiled_boundary_kernel(const __grid_constant__ StepParams<T> P, int two) {
  const Layout &L = P.L;
  const int X = blockIdx.x * blockDim.x + threadIdx.x;   // padded coordinates: ghosts are written too
  const int Y = blockIdx.y;
  const int z = blockIdx.z ? L.nz - 1 : 0;
  if (X >= L.px) return;
  if (blockIdx.z ? !P.out_hi : !P.jet_lo) return;
  const int x = ((X - GX) % L.nx + L.nx) % L.nx, y = ((Y - GY) % L.ny + L.ny) % L.ny;
  T o[NF_MAX];
  boundary_node<T>(P, P.in, x, y, z, P.step_next, o, two != 0);
  const long long i0 = ((long long)z * L.py + Y) * L.px + X;
  const int nf = two ? 11 : 10;
  for (int k = 0; k < nf; ++k) P.out.f[k][i0] = o[k];
}

template <typename T, int TX, int TY>
cudaError_t launch_tiled_t(TiledPlan &pl, const StepParams<T> &P, int src, int order, bool two, cudaStream_t st) {
  const bool slab = P.halo_lo || P.halo_hi;
  const TiledMaps &M = pl.maps[src];
  dim3 grid(M.ntx * M.nty, (P.L.nz + M.zc - 1) / M.zc);
  cudaError_t e = cudaSuccess;
#define TSLB_LAUNCH(ORD, TWOC, SL)                                                                      \
  do {                                                                                                \
    using Cf = TileCfg<T, TX, TY, TWOC>;                                                              \
    auto kern = tiled_step_kernel<T, TX, TY, ORD, TWOC, SL>;                                          \
    static bool attr_set = false;                                                                     \
    if (!attr_set) {                                                                                  \
      e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cf::SMEM_BYTES); \
      if (e != cudaSuccess) return e;                                                                 \
      attr_set = true;                                                                                \
    }                                                                                                 \
    kern<<<grid, Cf::NTHREADS, Cf::SMEM_BYTES, st>>>(P, M);                                           \
  } while (0)
  if (slab) {
    if (two) { if (order >= 3) TSLB_LAUNCH(3, true, true); else TSLB_LAUNCH(2, true, true); }
    else     { if (order >= 3) TSLB_LAUNCH(3, false, true); else TSLB_LAUNCH(2, false, true); }
  } else {
    if (two) { if (order >= 3) TSLB_LAUNCH(3, true, false); else TSLB_LAUNCH(2, true, false); }
    else     { if (order >= 3) TSLB_LAUNCH(3, false, false); else TSLB_LAUNCH(2, false, false); }
  }
#undef TSLB_LAUNCH
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (P.jet_lo || P.out_hi) {
    dim3 b(128), g((P.L.px + 127) / 128, P.L.py, 2);
    tiled_boundary_kernel<T><<<g, b, 0, st>>>(P, two ? 1 : 0);
    e = cudaGetLastError();
  }
  return e;
}

template <typename T>
cudaError_t launch_tiled(TiledPlan &pl, const StepParams<T> &P, int src, int order, bool two, cudaStream_t st);
template <>
inline cudaError_t launch_tiled<float>(TiledPlan &pl, const StepParams<float> &P, int src, int order, bool two, cudaStream_t st) {
  return launch_tiled_t<float, TSLB_F32_TX, TSLB_TY>(pl, P, src, order, two, st);
}
template <>
inline cudaError_t launch_tiled<double>(TiledPlan &pl, const StepParams<double> &P, int src, int order, bool two, cudaStream_t st) {
  return launch_tiled_t<double, TSLB_F64_TX, TSLB_TY>(pl, P, src, order, two, st);
}

}  // namespace tslb
