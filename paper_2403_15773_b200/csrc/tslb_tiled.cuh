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
//   x-pass  (segment 1)  K_abc (17 per node, recomputed for the pair's two x-neighbours)
//                        -> X^p_bc (24 per node), written to shared memory for tile rows +-1;
//   y-pass  (segment 2)  X^p_bc at rows y-1,y,y+1 -> Y^pq_c (18, registers);
//   z-push  (segment 2)  Y^pq_c of source plane k is pushed into the register accumulators of
//                        the destination planes k-1, k, k+1 (two live accumulator sets);
// so each stored moment is read from HBM once and the populations never exist in memory.
// The phase-field half (eqs. 20-24) runs in the same kernel from the phi ring:
// z-combinations of phi (aux warps), G and n = G/(|G|+eps) on tile+1 into a 3-plane ring,
// kappa = -div n, the kick, and the D3Q7 update assembled from per-plane fluxes -- phi, grad(phi),
// n and kappa never touch HBM.
//
// Thread roles: TY "compute" rows own the tile; 2 "aux" rows do the x-pass of the two halo rows,
// the phi z-combinations and the ring of the n field.  Two __syncthreads per plane.
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
  static constexpr int RY = TY + 2;        // staged moment rows y0-1 .. y0+TY
  static constexpr int RYP = TY + 4;       // staged phi rows y0-2 .. y0+TY+1
  static constexpr int S = 3;              // moment ring (planes k-1, k, k+1)
  static constexpr int SP = 4;             // phi ring
  static constexpr int NR = 3;             // ring of n / |G| planes
  static constexpr int NTHREADS = LX * RY;
  static constexpr int NAUX = 2 * LX;
  static constexpr int NX = 24;            // x-pass outputs per node
  static constexpr size_t al(size_t b) { return (b + 127) / 128 * 128; }
  static constexpr size_t MOM_BYTES = (size_t)10 * RY * RX * sizeof(T);   // one TMA box
  static constexpr size_t PHI_BYTES = (size_t)RYP * RX * sizeof(T);
  static constexpr size_t MOM_STAGE = al(MOM_BYTES);
  static constexpr size_t PHI_STAGE = al(PHI_BYTES);
  static constexpr size_t OFF_MOM = 0;
  static constexpr size_t OFF_PHI = OFF_MOM + S * MOM_STAGE;
  static constexpr size_t OFF_SZ = OFF_PHI + (TWO ? SP * PHI_STAGE : 0);
  static constexpr size_t OFF_DZ = OFF_SZ + (TWO ? PHI_STAGE : 0);
  static constexpr size_t NRM_PLANE = al((size_t)RY * RX * sizeof(T));
  static constexpr size_t OFF_NRM = OFF_DZ + (TWO ? PHI_STAGE : 0);
  static constexpr size_t GM_PLANE = al((size_t)TY * TX * sizeof(T));
  static constexpr size_t OFF_GM = OFF_NRM + (TWO ? NR * 3 * NRM_PLANE : 0);
  static constexpr size_t X_FIELD = al((size_t)RY * TX * sizeof(T));
  static constexpr size_t OFF_X = OFF_GM + (TWO ? NR * GM_PLANE : 0);
  static constexpr size_t OFF_BAR = OFF_X + NX * X_FIELD;
  static constexpr size_t SMEM_BYTES = OFF_BAR + 64;
};

struct TiledMaps {
  CUtensorMap mom;   // 4-D (px, py, nz, 10) over the SOURCE buffer, box (RX, RY, 1, 10)
  CUtensorMap phi;   // 3-D (px, py, nz) over the source phi, box (RX, RYP, 1)
  int ntx, nty;      // tiles per row / column
  int zc;            // planes per z chunk
};

// 1-D three-point operators of the tensor-product basis, un-normalised input coefficient of
// Hermite index U, output moment of Hermite index W, acting on P = g(-1)+g(+1) side sums
// (P = g(x-1)+g(x+1), Q = g(x-1)-g(x+1), C = g(x)); table derived in DESIGN.md §6:
//   U=0: W0: P/6+2C/3   W1: Q/6   W2: P/9-2C/9
//   U=1: W0: Q/2        W1: P/2   W2: Q/3
//   U=2: W0: P/2-C      W1: Q/2   W2: (P+C)/3
template <int U, int W, typename V, typename T>
__device__ __forceinline__ V op_acc(V acc, V Pv, V Qv, V Cv) {
  if (U == 0 && W == 0) return pfma(Cv, T(2.0 / 3.0), pfma(Pv, T(1.0 / 6.0), acc));
  if (U == 0 && W == 1) return pfma(Qv, T(1.0 / 6.0), acc);
  if (U == 0 && W == 2) return pfma(Cv, T(-2.0 / 9.0), pfma(Pv, T(1.0 / 9.0), acc));
  if (U == 1 && W == 0) return pfma(Qv, T(0.5), acc);
  if (U == 1 && W == 1) return pfma(Pv, T(0.5), acc);
  if (U == 1 && W == 2) return pfma(Qv, T(1.0 / 3.0), acc);
  if (U == 2 && W == 0) return pfma(Pv, T(0.5), acc - Cv);
  if (U == 2 && W == 1) return pfma(Qv, T(0.5), acc);
  return pfma(Pv + Cv, T(1.0 / 3.0), acc);
}

template <typename T> __device__ __forceinline__ Pair<T> prcp(Pair<T> a);
template <> __device__ __forceinline__ F2 prcp<float>(F2 a) { return F2(__frcp_rn(a.x), __frcp_rn(a.y)); }
template <> __device__ __forceinline__ D2 prcp<double>(D2 a) { return D2(1.0 / a.x, 1.0 / a.y); }

__device__ __forceinline__ float rcp1(float s) { return __frcp_rn(s); }
__device__ __forceinline__ double rcp1(double s) { return 1.0 / s; }

// ------------------------------------------------------------------ the kernel
template <typename T, int TX, int TY, int ORDER, bool TWO>
__global__ void __launch_bounds__((TX / 2) * (TY + 2), 1)
tiled_step_kernel(const __grid_constant__ StepParams<T> P, const __grid_constant__ TiledMaps M) {
  using C = TileCfg<T, TX, TY, TWO>;
  using V = Pair<T>;
  constexpr int LX = C::LX, HL = C::HL, RX = C::RX, RY = C::RY, RYP = C::RYP, S = C::S, SP = C::SP, NR = C::NR;
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::OFF_BAR);
  auto mom_at = [&](int slot, int f) { return reinterpret_cast<T *>(smem + C::OFF_MOM + slot * C::MOM_STAGE) + (size_t)f * RY * RX; };
  auto phi_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_PHI + slot * C::PHI_STAGE); };
  auto nrm_at = [&](int slot, int comp) { return reinterpret_cast<T *>(smem + C::OFF_NRM + (slot * 3 + comp) * C::NRM_PLANE); };
  auto gm_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_GM + slot * C::GM_PLANE); };
  auto x_at = [&](int f) { return reinterpret_cast<T *>(smem + C::OFF_X + f * C::X_FIELD); };
  T *s_sz = reinterpret_cast<T *>(smem + C::OFF_SZ);
  T *s_dz = reinterpret_cast<T *>(smem + C::OFF_DZ);

  const Layout &L = P.L;
  const int t = threadIdx.x;
  const int lx = t % LX;
  const int tr = t / LX;
  const bool aux = tr >= TY;
  const int r = aux ? (tr == TY ? 0 : RY - 1) : tr + 1;   // region row (y = y0 - 1 + r)
  const int c0 = HL + 2 * lx;                              // staged column of the pair's first node
  const int x0 = (blockIdx.x % M.ntx) * TX;
  const int y0 = (blockIdx.x / M.ntx) * TY;
  const int z0 = blockIdx.y * M.zc;
  const int z1 = min(z0 + M.zc, L.nz);
  const int kb = z0 - 1;                 // first source plane
  const int NG = z1 - kb + 1;            // load groups / x-pass planes: kb .. z1
  const int NI = NG + 1;                 // iterations

  auto zmap = [&](int z) {
    if (P.zper) { z %= L.nz; return z < 0 ? z + L.nz : z; }
    return z < 0 ? 0 : (z >= L.nz ? L.nz - 1 : z);
  };
  // group g (relative index): moments of plane kb+g -> slot g%S, phi of plane kb+g+1 -> slot (g+2)%SP
  auto issue = [&](int g) {
    uint64_t *bar = &bars[g % S];
    uint32_t bytes = (uint32_t)C::MOM_BYTES + (TWO ? (uint32_t)C::PHI_BYTES : 0u);
    if (TWO && g == 0) bytes += 2u * (uint32_t)C::PHI_BYTES;
    mbar_expect_tx(bar, bytes);
    tma_load_4d(mom_at(g % S, 0), &M.mom, bar, x0 - HL + GX, y0 - 1 + GY, zmap(kb + g), 0);
    if (TWO) {
      tma_load_3d(phi_at((g + 2) % SP), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb + g + 1));
      if (g == 0) {
        tma_load_3d(phi_at(0), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb - 1));
        tma_load_3d(phi_at(1), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb));
      }
    }
  };

#if defined(TSLB_DBG) && TSLB_DBG == 5
  return;
#endif
  if (t == 0) {
    for (int s = 0; s < S; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
#if defined(TSLB_DBG) && TSLB_DBG == 4
  return;
#endif
  if (t == 0) {
    issue(0);
    if (NG > 1) issue(1);
  }

  const V omc(P.omc);
  V accA[10], accB[10];     // Hermite moments being accumulated for planes k and k+1
  V fl[10];                 // finished flow part of the plane completed in the previous iteration:
                            // drho', u_b (3), Pi^neq' (6)
  V c_inpl(T(0)), c_upa(T(0)), c_upb(T(0));
#pragma unroll
  for (int m = 0; m < 10; ++m) { accA[m] = V(T(0)); accB[m] = V(T(0)); fl[m] = V(T(0)); }

  for (int i = 0; i < NI; ++i) {
    const int k = kb + i;
#if defined(TSLB_DBG) && TSLB_DBG == 1
    return;
#endif
    if (i < NG) mbar_wait(&bars[i % S], (uint32_t)((i / S) & 1));
#if defined(TSLB_DBG) && TSLB_DBG == 2
    __syncthreads(); return;
#endif

    // =========================== segment 1 ===========================
    if (TWO && aux && i < NG) {
      // A1: z-combinations of phi for plane k: sz = S_z phi, dz = delta_z phi on the phi halo region
      const T *pm = phi_at(i % SP), *pc = phi_at((i + 1) % SP), *pp = phi_at((i + 2) % SP);
      const int ia = (tr - TY) * LX + lx;
      for (int e = ia; e < RYP * RX / 2; e += C::NAUX) {
        const V a = lds_pair(pm + 2 * e), b = lds_pair(pc + 2 * e), c = lds_pair(pp + 2 * e);
        sts_pair(s_sz + 2 * e, pfma(b, T(2.0 / 3.0), (a + c) * T(1.0 / 6.0)));
        sts_pair(s_dz + 2 * e, (c - a) * T(0.5));
      }
    }
    if (i < NG) {
      // A2: x-pass of region row r of plane k.  A = nodes (x-1, x), B = nodes (x+1, x+2).
      V KA[NK], KB[NK];
      {
        V mA[10], mB[10];
#pragma unroll
        for (int f = 0; f < 10; ++f) {
          const T *p = mom_at(i % S, f) + r * RX + c0;
          const V own = lds_pair(p);
          mA[f] = V(p[-1], own.x);
          mB[f] = V(own.y, p[2]);
        }
        hermite_coeffs<ORDER, V>(mA[0], mA[1], mA[2], mA[3], mA[4], mA[5], mA[6], mA[7], mA[8], mA[9], omc, KA);
        hermite_coeffs<ORDER, V>(mB[0], mB[1], mB[2], mB[3], mB[4], mB[5], mB[6], mB[7], mB[8], mB[9], omc, KB);
      }
      // groups (b,c) -> K indices for a = 0,1,2 (-1: absent)
      constexpr int GA[8][3] = {{K000, K100, K200}, {K010, K110, K210}, {K001, K101, K201}, {K020, K120, -1},
                                {K002, K102, -1},   {K011, K111, -1},   {K021, -1, -1},     {K012, -1, -1}};
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        V X0(T(0)), X1(T(0)), X2(T(0));
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          if (GA[g][a] < 0) continue;
          const V ka = KA[GA[g][a]], kbv = KB[GA[g][a]];
          const V Pv = ka + kbv, Qv = ka - kbv, Cv(ka.y, kbv.x);
          if (a == 0) { X0 = op_acc<0, 0, V, T>(X0, Pv, Qv, Cv); X1 = op_acc<0, 1, V, T>(X1, Pv, Qv, Cv); X2 = op_acc<0, 2, V, T>(X2, Pv, Qv, Cv); }
          if (a == 1) { X0 = op_acc<1, 0, V, T>(X0, Pv, Qv, Cv); X1 = op_acc<1, 1, V, T>(X1, Pv, Qv, Cv); X2 = op_acc<1, 2, V, T>(X2, Pv, Qv, Cv); }
          if (a == 2) { X0 = op_acc<2, 0, V, T>(X0, Pv, Qv, Cv); X1 = op_acc<2, 1, V, T>(X1, Pv, Qv, Cv); X2 = op_acc<2, 2, V, T>(X2, Pv, Qv, Cv); }
        }
        sts_pair(x_at(3 * g + 0) + r * TX + 2 * lx, X0);
        sts_pair(x_at(3 * g + 1) + r * TX + 2 * lx, X1);
        sts_pair(x_at(3 * g + 2) + r * TX + 2 * lx, X2);
      }
    }
    if (!aux && i >= 1) {
      V phin(T(0)), ukx(T(0)), uky(T(0)), ukz(T(0));
      const int j = k - 2;                         // plane finalised in this iteration
      const bool fin = (j >= z0);                  // (j < z1 always: k <= z1 + 1)
      if (TWO) {
        // fluxes of plane k-1 (all operands resident: moments slot (i-1)%S, phi slot i%SP, n slot (i-1)%NR)
        const int ms = (i - 1) % S, ns = (i - 1) % NR;
        const T *ph = phi_at(i % SP) + (r + 1) * RX + c0;
        const T gam = P.gamma;
        auto gplus = [&](T p, T u, T n) { return p * (T(1) + T(4) * u) + gam * p * (T(1) - p) * n; };
        auto gminus = [&](T p, T u, T n) { return p * (T(1) - T(4) * u) - gam * p * (T(1) - p) * n; };
        // x direction: columns c0-1 .. c0+2
        const T *uxp = mom_at(ms, F_UX) + r * RX + c0;
        const T *nxp = nrm_at(ns, 0) + r * RX + c0;
        const V phc = lds_pair(ph), uxc = lds_pair(uxp), nxc = lds_pair(nxp);
        V inpl;
        inpl.x = gplus(ph[-1], uxp[-1], nxp[-1]) + gminus(phc.y, uxc.y, nxc.y);
        inpl.y = gplus(phc.x, uxc.x, nxc.x) + gminus(ph[2], uxp[2], nxp[2]);
        // y direction: rows r-1 (south, c_i = +e_y) and r+1 (north)
        const T *uyp = mom_at(ms, F_UY) + r * RX + c0;
        const T *nyp = nrm_at(ns, 1) + r * RX + c0;
        const V phs = lds_pair(ph - RX), uys = lds_pair(uyp - RX), nys = lds_pair(nyp - RX);
        const V phn_ = lds_pair(ph + RX), uyn = lds_pair(uyp + RX), nyn = lds_pair(nyp + RX);
        inpl.x += gplus(phs.x, uys.x, nys.x) + gminus(phn_.x, uyn.x, nyn.x);
        inpl.y += gplus(phs.y, uys.y, nys.y) + gminus(phn_.y, uyn.y, nyn.y);
        inpl.x = T(0.25) * phc.x + T(0.125) * inpl.x;
        inpl.y = T(0.25) * phc.y + T(0.125) * inpl.y;
        // z direction: this plane's contribution to the planes above (up) and below (down)
        const V uzc = lds_pair(mom_at(ms, F_UZ) + r * RX + c0), nzc = lds_pair(nrm_at(ns, 2) + r * RX + c0);
        const V up(gplus(phc.x, uzc.x, nzc.x), gplus(phc.y, uzc.y, nzc.y));
        const V down(gminus(phc.x, uzc.x, nzc.x), gminus(phc.y, uzc.y, nzc.y));
        if (fin) {
          // a7: phi'(j) = inpl(j) + up(j-1)/8 + down(j+1)/8       (eqs. 23-24)
          phin = pfma(c_upa + down, T(0.125), c_inpl);
          // a5: kappa(j) = -div n over the 27-point stencil, n planes j-1, j, j+1
          const int sm_ = (i + NR - 3) % NR, s0 = (i + NR - 2) % NR, sp_ = (i + NR - 1) % NR;
          const T w1 = T(1.0 / 6.0), w0 = T(2.0 / 3.0);
          V kap(T(0));
          {
            // d/dx of S_y S_z n_x
            V own(T(0)), nb(T(0));
            const int sl[3] = {sm_, s0, sp_};
#pragma unroll
            for (int dz = 0; dz < 3; ++dz)
#pragma unroll
              for (int dy = -1; dy <= 1; ++dy) {
                const T w = (dz == 1 ? w0 : w1) * (dy == 0 ? w0 : w1);
                const T *q = nrm_at(sl[dz], 0) + (r + dy) * RX + c0;
                own = pfma(lds_pair(q), w, own);
                nb = pfma(V(q[-1], q[2]), w, nb);
              }
            kap.x += T(0.5) * (own.y - nb.x);
            kap.y += T(0.5) * (nb.y - own.x);
            // d/dy of S_x S_z n_y
            V dO(T(0)), dN(T(0));
#pragma unroll
            for (int dz = 0; dz < 3; ++dz) {
              const T w = (dz == 1 ? w0 : w1);
              const T *qn = nrm_at(sl[dz], 1) + (r + 1) * RX + c0;
              const T *qs = nrm_at(sl[dz], 1) + (r - 1) * RX + c0;
              dO = pfma(lds_pair(qn) - lds_pair(qs), w, dO);
              dN = pfma(V(qn[-1], qn[2]) - V(qs[-1], qs[2]), w, dN);
            }
            kap.x += T(0.5) * (w1 * dN.x + w0 * dO.x + w1 * dO.y);
            kap.y += T(0.5) * (w1 * dO.x + w0 * dO.y + w1 * dN.y);
            // d/dz of S_x S_y n_z
            V eO(T(0)), eN(T(0));
#pragma unroll
            for (int dy = -1; dy <= 1; ++dy) {
              const T w = (dy == 0 ? w0 : w1);
              const T *qp = nrm_at(sp_, 2) + (r + dy) * RX + c0;
              const T *qm = nrm_at(sm_, 2) + (r + dy) * RX + c0;
              eO = pfma(lds_pair(qp) - lds_pair(qm), w, eO);
              eN = pfma(V(qp[-1], qp[2]) - V(qm[-1], qm[2]), w, eN);
            }
            kap.x += T(0.5) * (w1 * eN.x + w0 * eO.x + w1 * eO.y);
            kap.y += T(0.5) * (w1 * eO.x + w0 * eO.y + w1 * eN.y);
          }
          // a6: F = sigma kappa G, G = n (|G| + eps); u' = u_b + F / rho'   (kappa = -div: sign below)
          const V gm = lds_pair(gm_at(s0) + tr * TX + 2 * lx) + V(T(1e-12));
          const V rinv = prcp<T>(fl[0] + V(T(1)));
          const V sc = (kap * gm) * rinv * (-P.sigma);
          ukx = lds_pair(nrm_at(s0, 0) + r * RX + c0) * sc;
          uky = lds_pair(nrm_at(s0, 1) + r * RX + c0) * sc;
          ukz = lds_pair(nrm_at(s0, 2) + r * RX + c0) * sc;
        }
        c_upa = c_upb; c_upb = up; c_inpl = inpl;
      }
      if (fin && (P.zper || (j > 0 && j < L.nz - 1))) {
        // a9: store plane j (and its periodic ghost images)
        const int x = x0 + 2 * lx, y = y0 + tr;
        V o[NF_MAX];
        o[0] = fl[0];
        o[1] = fl[1] + ukx; o[2] = fl[2] + uky; o[3] = fl[3] + ukz;
#pragma unroll
        for (int m = 4; m < 10; ++m) o[m] = fl[m];
        o[10] = phin;
        const int xg = x < 2 ? x + L.nx : (x >= L.nx - 2 ? x - L.nx : x);
        const int yg = y < GY ? y + L.ny : (y >= L.ny - GY ? y - L.ny : y);
        const long long i00 = L.idx(x, y, j), i10 = L.idx(xg, y, j), i01 = L.idx(x, yg, j), i11 = L.idx(xg, yg, j);
#pragma unroll
        for (int m = 0; m < (TWO ? 11 : 10); ++m) {
          T *base = P.out.f[m];
          *reinterpret_cast<V *>(base + i00) = o[m];
          if (xg != x) *reinterpret_cast<V *>(base + i10) = o[m];
          if (yg != y) {
            *reinterpret_cast<V *>(base + i01) = o[m];
            if (xg != x) *reinterpret_cast<V *>(base + i11) = o[m];
          }
        }
      }
    }
    __syncthreads();
#if defined(TSLB_DBG) && TSLB_DBG == 3
    return;
#endif
    if (t == 0 && i + 2 < NG) issue(i + 2);

    // =========================== segment 2 ===========================
    if (i < NG) {
      if (!aux) {
        // B2: y-pass (rows r-1, r, r+1 of X) and z-push into the accumulators.
        // X field of group (b,c) and x-moment p is 3*g + p with g as in GA above:
        //   c = 0: b = 0,1,2 -> g = 0,1,3;  c = 1: b = 0,1,2 -> g = 2,5,6;  c = 2: b = 0,1 -> g = 4,7
        constexpr int GB[3][3] = {{0, 1, 3}, {2, 5, 6}, {4, 7, -1}};
        V outm[10];
#pragma unroll
        for (int m = 0; m < 10; ++m) outm[m] = accA[m];
        // moment index of (p,q,rr)
        constexpr int MI[3][3][3] = {{{0, 3, 6}, {2, 9, -1}, {5, -1, -1}}, {{1, 8, -1}, {7, -1, -1}, {-1, -1, -1}}, {{4, -1, -1}, {-1, -1, -1}, {-1, -1, -1}}};
#pragma unroll
        for (int p = 0; p < 3; ++p) {
          V Yq[3][3];   // [q][c]
#pragma unroll
          for (int q = 0; q < 3; ++q)
#pragma unroll
            for (int c = 0; c < 3; ++c) Yq[q][c] = V(T(0));
#pragma unroll
          for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int b = 0; b < 3; ++b) {
              if (GB[c][b] < 0) continue;
              const T *xp = x_at(3 * GB[c][b] + p) + r * TX + 2 * lx;
              const V gs = lds_pair(xp - TX), gc = lds_pair(xp), gn = lds_pair(xp + TX);
              const V Pv = gs + gn, Qv = gs - gn;
              if (b == 0) { Yq[0][c] = op_acc<0, 0, V, T>(Yq[0][c], Pv, Qv, gc); if (p <= 1) Yq[1][c] = op_acc<0, 1, V, T>(Yq[1][c], Pv, Qv, gc); if (p == 0) Yq[2][c] = op_acc<0, 2, V, T>(Yq[2][c], Pv, Qv, gc); }
              if (b == 1) { Yq[0][c] = op_acc<1, 0, V, T>(Yq[0][c], Pv, Qv, gc); if (p <= 1) Yq[1][c] = op_acc<1, 1, V, T>(Yq[1][c], Pv, Qv, gc); if (p == 0) Yq[2][c] = op_acc<1, 2, V, T>(Yq[2][c], Pv, Qv, gc); }
              if (b == 2) { Yq[0][c] = op_acc<2, 0, V, T>(Yq[0][c], Pv, Qv, gc); if (p <= 1) Yq[1][c] = op_acc<2, 1, V, T>(Yq[1][c], Pv, Qv, gc); if (p == 0) Yq[2][c] = op_acc<2, 2, V, T>(Yq[2][c], Pv, Qv, gc); }
            }
#pragma unroll
          for (int q = 0; q + p <= 2; ++q) {
            const V Y0 = Yq[q][0], Y1 = Yq[q][1], Y2 = Yq[q][2];
            const V h = pfma(Y0, T(1.0 / 6.0), Y2 * T(0.5));
            const V ap = pfma(Y1, T(0.5), h);      // -> plane k+1
            const V am = pfma(Y1, T(-0.5), h);     // -> plane k-1
            const V a0 = pfma(Y0, T(2.0 / 3.0), V(T(0)) - Y2);   // -> plane k
            {
              const int m = MI[p][q][0];
              outm[m] = outm[m] + am; accA[m] = accB[m] + a0; accB[m] = ap;
            }
            if (p + q <= 1) {
              const int m = MI[p][q][1];
              outm[m] = outm[m] - am; accA[m] = accB[m]; accB[m] = ap;
            }
            if (p + q == 0) {
              const int m = MI[p][q][2];
              outm[m] = pfma(am, T(2.0 / 3.0), outm[m]);
              accA[m] = pfma(a0, T(-1.0 / 3.0), accB[m]);
              accB[m] = ap * T(2.0 / 3.0);
            }
          }
        }
        // a4: plane k-1 is complete: u_b = m'/rho', Pi^neq' = Pi' - rho' u_b u_b (Hermite form)
        const V inv = prcp<T>(outm[0] + V(T(1)));
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
        // B1: G = grad(phi), n = G/(|G|+eps) of plane k on tile+1 -> ring slot i%NR
        auto gn_pair = [&](int rr, int c, bool write_gm) {
          // columns c-1 .. c+2 (clamped at the staged edge; edge results are never used)
          const int cl = c > 0 ? c - 1 : 0, cr = c + 2 < RX ? c + 2 : RX - 1;
          const int rp = rr + 1;
          T Tc[4], Uc[4], Vc[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int cc = q == 0 ? cl : (q == 3 ? cr : c + q - 1);
            const T s_m = s_sz[(rp - 1) * RX + cc], s_0 = s_sz[rp * RX + cc], s_p = s_sz[(rp + 1) * RX + cc];
            const T d_m = s_dz[(rp - 1) * RX + cc], d_0 = s_dz[rp * RX + cc], d_p = s_dz[(rp + 1) * RX + cc];
            Tc[q] = T(1.0 / 6.0) * (s_m + s_p) + T(2.0 / 3.0) * s_0;
            Uc[q] = T(0.5) * (s_p - s_m);
            Vc[q] = T(1.0 / 6.0) * (d_m + d_p) + T(2.0 / 3.0) * d_0;
          }
          T g[2][3];
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            g[e][0] = T(0.5) * (Tc[e + 2] - Tc[e]);
            g[e][1] = T(1.0 / 6.0) * (Uc[e] + Uc[e + 2]) + T(2.0 / 3.0) * Uc[e + 1];
            g[e][2] = T(1.0 / 6.0) * (Vc[e] + Vc[e + 2]) + T(2.0 / 3.0) * Vc[e + 1];
          }
          const T s0_ = g[0][0] * g[0][0] + g[0][1] * g[0][1] + g[0][2] * g[0][2];
          const T s1_ = g[1][0] * g[1][0] + g[1][1] * g[1][1] + g[1][2] * g[1][2];
          const T m0_ = tsqrt<T>(s0_), m1_ = tsqrt<T>(s1_);                    // |G|
          const T i0_ = rcp1(m0_ + T(1e-12)), i1_ = rcp1(m1_ + T(1e-12));     // 1/(|G|+eps), reading A7
          const int slot = i % NR;
#pragma unroll
          for (int a = 0; a < 3; ++a) sts_pair(nrm_at(slot, a) + rr * RX + c, V(g[0][a] * i0_, g[1][a] * i1_));
          if (write_gm) sts_pair(gm_at(slot) + (rr - 1) * TX + (c - HL), V(m0_, m1_));
        };
        if (!aux) {
          gn_pair(r, c0, true);
        } else {
          const int ia = (tr - TY) * LX + lx;
          constexpr int PPR = TX / 2 + 2;                // pairs per full ring row: cols HL-2 .. HL+TX+1
          constexpr int NT = 2 * PPR + 2 * TY;           // ring tasks
          for (int e = ia; e < NT; e += C::NAUX) {
            int rr, c;
            if (e < 2 * PPR) { rr = (e < PPR) ? 0 : RY - 1; c = HL - 2 + 2 * (e % PPR); }
            else { const int q = e - 2 * PPR; rr = 1 + (q >> 1); c = (q & 1) ? HL + TX : HL - 2; }
            gn_pair(rr, c, false);
          }
        }
      }
    }
    __syncthreads();
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

// tile shapes: fp32 64x8, fp64 32x8 (same bytes per row)
#ifndef TSLB_F32_TX
#define TSLB_F32_TX 64
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
  return nx % tx == 0 && ny % ty == 0 && nz >= 1 && nx >= tx && ny >= ty;
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
    cuuint64_t gdim[4] = {(cuuint64_t)L.px, (cuuint64_t)L.py, (cuuint64_t)L.nz, 10};
    cuuint64_t gstr[3] = {(cuuint64_t)L.px * es, (cuuint64_t)L.plane * es, (cuuint64_t)fstride};
    cuuint32_t box[4] = {(cuuint32_t)RX, (cuuint32_t)RY, 1, 10};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(&pl.maps[b].mom, dt, 4, fields[b][0], gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled(moments) failed: " + std::to_string((int)r); return false; }
    if (pl.two) {
      cuuint32_t boxp[3] = {(cuuint32_t)RX, (cuuint32_t)RYP, 1};
      r = enc(&pl.maps[b].phi, dt, 3, fields[b][F_PHI], gdim, gstr, boxp, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) { why = "cuTensorMapEncodeTiled(phi) failed: " + std::to_string((int)r); return false; }
    } else {
      pl.maps[b].phi = pl.maps[b].mom;
    }
    pl.maps[b].ntx = L.nx / pl.tx;
    pl.maps[b].nty = L.ny / pl.ty;
  }
  // z chunking: enough CTAs to fill the machine several times, chunks long enough to amortise the
  // 3-plane pipeline prologue
  const long long tiles = (long long)(L.nx / pl.tx) * (L.ny / pl.ty);
  int zc = 128;
  while (zc > 8 && tiles * ((L.nz + zc - 1) / zc) < 4 * 148) zc /= 2;
  if (zc > L.nz) zc = L.nz;
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
  const int x = ((X - GX) % L.nx + L.nx) % L.nx, y = ((Y - GY) % L.ny + L.ny) % L.ny;
  T o[NF_MAX];
  boundary_node<T>(P, P.in, x, y, z, P.step_next, o, two != 0);
  const long long i0 = ((long long)z * L.py + Y) * L.px + X;
  const int nf = two ? 11 : 10;
  for (int k = 0; k < nf; ++k) P.out.f[k][i0] = o[k];
}

template <typename T, int TX, int TY>
cudaError_t launch_tiled_t(TiledPlan &pl, const StepParams<T> &P, int src, int order, bool two, cudaStream_t st) {
  const TiledMaps &M = pl.maps[src];
  dim3 grid(M.ntx * M.nty, (P.L.nz + M.zc - 1) / M.zc);
  cudaError_t e = cudaSuccess;
#define TSLB_LAUNCH(ORD, TWOC)                                                                        \
  do {                                                                                                \
    using Cf = TileCfg<T, TX, TY, TWOC>;                                                              \
    auto kern = tiled_step_kernel<T, TX, TY, ORD, TWOC>;                                              \
    static bool attr_set = false;                                                                     \
    if (!attr_set) {                                                                                  \
      e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cf::SMEM_BYTES); \
      if (e != cudaSuccess) return e;                                                                 \
      attr_set = true;                                                                                \
    }                                                                                                 \
    kern<<<grid, Cf::NTHREADS, Cf::SMEM_BYTES, st>>>(P, M);                                           \
  } while (0)
  if (two) { if (order >= 3) TSLB_LAUNCH(3, true); else TSLB_LAUNCH(2, true); }
  else     { if (order >= 3) TSLB_LAUNCH(3, false); else TSLB_LAUNCH(2, false); }
#undef TSLB_LAUNCH
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (!P.zper) {
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
