// tslb_tiled_ws.cuh -- warp-specialised variant of the tiled kernel (fp32, two-component).
//
// Same tile, same staging, same mathematics and the same two barriers per plane as
// tiled_step_kernel (tslb_tiled.cuh), but every node pair is served by TWO threads that run
// concurrently instead of one thread doing both jobs back to back:
//   flow  warps 0-3  x-pass, y-push, y-pull, z-push into the register accumulators, rho', u_b,
//                    Pi^neq'; they store rho' and Pi^neq' and hand u_b and 1/rho' to the phase thread;
//   phase warps 4-7  T/U/V pre-combinations, G, n, z-combined n, kappa, the kick, the D3Q7 fluxes,
//                    phi'; they store u' and phi';
//   aux   warp  8    x-pass of the two halo rows, x-pass terms of the two halo columns.
// The tiled kernel is latency-bound at 12 warps/SM because one thread carries ~100 persistent
// registers; splitting the state lets 18 warps/SM run (2 CTAs x 9 warps) with the register file
// re-divided by setmaxnreg: flow 152, phase 72, aux 112 registers per thread.
#pragma once
#include "tslb_tiled.cuh"

namespace tslb {

template <int TX, int TY>
struct WsCfg {
  using C = TileCfg<float, TX, TY, true>;
  static constexpr int LX = C::LX;
  static constexpr int NFLOW = LX * TY;              // flow threads  (= phase threads)
  static constexpr int NTHREADS = 2 * NFLOW + 32;    // + one aux warp
  static constexpr size_t OFF_FL = C::OFF_BAR + 64;  // u_b (3) and 1/rho' of the completed plane
  static constexpr size_t FL_FIELD = (size_t)TY * TX * sizeof(float);
  static constexpr size_t SMEM_BYTES = OFF_FL + 4 * FL_FIELD;
  static_assert(NFLOW == 128, "warp-group register re-allocation needs 4 flow and 4 phase warps");
};

template <int TX, int TY, int ORDER>
__global__ void __launch_bounds__(WsCfg<TX, TY>::NTHREADS, 2)
tiled_ws_kernel(const __grid_constant__ StepParams<float> P, const __grid_constant__ TiledMaps M) {
  using T = float;
  using W = WsCfg<TX, TY>;
  using C = typename W::C;
  using V = Pair<T>;
  constexpr int LX = C::LX, HL = C::HL, RX = C::RX, RY = C::RY, S = C::S, SP = C::SP, NR = C::NR;
  constexpr int PL = (int)(C::PLANE / sizeof(T));
  constexpr int YPF = (int)(C::YP_FIELD / sizeof(T));
  constexpr int MF = RY * RX;
  constexpr int FLF = TY * TX;
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::OFF_BAR);
  auto mom_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_MOM + slot * C::MOM_STAGE); };
  auto phi_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_PHI + slot * C::PHI_STAGE); };
  auto nrm_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_NRM + slot * 3 * C::PLANE); };
  T *s_tuv = reinterpret_cast<T *>(smem + C::OFF_TUV);
  T *s_zc = reinterpret_cast<T *>(smem + C::OFF_ZC);
  T *s_ap = reinterpret_cast<T *>(smem + C::OFF_AP);
  T *s_am = reinterpret_cast<T *>(smem + C::OFF_AM);
  T *s_xhl = reinterpret_cast<T *>(smem + C::OFF_XH);
  T *s_xhr = s_xhl + 8 * RY;
  T *s_fl = reinterpret_cast<T *>(smem + W::OFF_FL);

  const Layout &L = P.L;
  const int t = threadIdx.x;
  const int role = t < W::NFLOW ? 0 : (t < 2 * W::NFLOW ? 1 : 2);   // flow / phase / aux
  const int tt = t - role * W::NFLOW;                                // index inside the role
  const int lx = tt % LX;
  const int tr = tt / LX;                                            // tile row (flow, phase)
  const int r = role == 2 ? (tr == 0 ? 0 : RY - 1) : tr + 1;        // region row
  const int c0 = HL + 2 * lx;
  const int oM = r * RX + c0;
  const int oY = r * TX + 2 * lx;
  const int oF = tr * TX + 2 * lx;                                   // offset in an FL field
  // x-exchange word: word (t & 31) of the y-push row owned by lane 0 of the warp
  const int oX = (role == 2 ? 0 : ((tt & ~31) / LX) + 1) * TX + (t & 31);
  const int x0 = (blockIdx.x % M.ntx) * TX;
  const int y0 = (blockIdx.x / M.ntx) * TY;
  const int z0 = blockIdx.y * M.zc;
  const int z1 = min(z0 + M.zc, L.nz);
  const int kb = z0 - 1;
  const int NG = z1 - kb + 1;
  const int NI = NG + 1;

  auto zmap = [&](int z) {
    if (P.zper) { while (z < 0) z += L.nz; while (z >= L.nz) z -= L.nz; return z; }
    return z < 0 ? 0 : (z >= L.nz ? L.nz - 1 : z);
  };
  auto issue = [&](int g) {
    uint64_t *bar = &bars[g % S];
    uint32_t bytes = (uint32_t)C::MOM_BYTES + (uint32_t)C::PHI_BYTES;
    if (g == 0) bytes += 2u * (uint32_t)C::PHI_BYTES;
    mbar_expect_tx(bar, bytes);
    tma_load_4d(mom_at(g % S), &M.mom, bar, x0 - HL + GX, y0 - 1 + GY, zmap(kb + g), 0);
    tma_load_3d(phi_at((g + 2) % SP), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb + g + 1));
    if (g == 0) {
      tma_load_3d(phi_at(0), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb - 1));
      tma_load_3d(phi_at(1), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(kb));
    }
  };

  if (t == 0) {
    for (int s = 0; s < S; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (t == 0) {
    issue(0);
    if (NG > 1) issue(1);
  }

  const V omc(P.omc);
  const T w1 = T(1.0 / 6.0), w0 = T(2.0 / 3.0);

  // global store offsets of the pair (plane 0) and of its periodic ghost images
  const int gx_ = x0 + 2 * lx, gy_ = y0 + tr;
  const int gxg = gx_ < 2 ? gx_ + L.nx : (gx_ >= L.nx - 2 ? gx_ - L.nx : gx_);
  const int gyg = gy_ < GY ? gy_ + L.ny : (gy_ >= L.ny - GY ? gy_ - L.ny : gy_);
  const long long o00 = L.idx(gx_, gy_, 0), o10 = L.idx(gxg, gy_, 0), o01 = L.idx(gx_, gyg, 0), o11 = L.idx(gxg, gyg, 0);
  const bool edge = gxg != gx_ || gyg != gy_;
  auto store_ghosts = [&](int m, long long zo, V v) {
    T *base = P.out.f[m] + zo;
    if (gxg != gx_) *reinterpret_cast<V *>(base + o10) = v;
    if (gyg != gy_) {
      *reinterpret_cast<V *>(base + o01) = v;
      if (gxg != gx_) *reinterpret_cast<V *>(base + o11) = v;
    }
  };

  // x-pass of region row r of the plane in moment slot ms, then the y-push terms (flow and aux)
  auto xpass = [&](int ms, V *A0) {
    V Xg[8][3];
    {
      V m[10], K[NK];
      const T *p = mom_at(ms) + oM;
#pragma unroll
      for (int f = 0; f < 10; ++f) m[f] = lds_pair(p + f * MF);
      hermite_coeffs<ORDER, V>(m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], m[8], m[9], omc, K);
      V gp[8], gm[8], g0[8];
      push3<3, V, T>(K[K000], K[K100], K[K200], gp[0], gm[0], g0[0]);
      push3<3, V, T>(K[K010], K[K110], K[K210], gp[1], gm[1], g0[1]);
      push3<2, V, T>(K[K020], K[K120], K[K120], gp[2], gm[2], g0[2]);
      push3<3, V, T>(K[K001], K[K101], K[K201], gp[3], gm[3], g0[3]);
      push3<2, V, T>(K[K011], K[K111], K[K111], gp[4], gm[4], g0[4]);
      push3<1, V, T>(K[K021], K[K021], K[K021], gp[5], gm[5], g0[5]);
      push3<2, V, T>(K[K002], K[K102], K[K102], gp[6], gm[6], g0[6]);
      push3<1, V, T>(K[K012], K[K012], K[K012], gp[7], gm[7], g0[7]);
      T *xp = s_ap + oX, *xm = s_am + oX;
#pragma unroll
      for (int g = 0; g < 8; ++g) { xp[g * YPF] = gp[g].y; xm[g * YPF] = gm[g].x; }
      __syncwarp();
      const T *pl = lx == 0 ? s_xhl + r : xp - 1, *pr = lx == LX - 1 ? s_xhr + r : xm + 1;
      const int sl = lx == 0 ? RY : YPF, sr = lx == LX - 1 ? RY : YPF;
#pragma unroll
      for (int g = 0; g < 8; ++g)
        pull3s<V, T>(pl[g * sl], gp[g].x, gm[g].y, pr[g * sr], g0[g], Xg[g][0], Xg[g][1], Xg[g][2]);
      __syncwarp();
    }
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
  };

  if (role == 0) {
    // ======================================= flow threads =======================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 128;");
    V accA[10], accB[10], A0[9];
#pragma unroll
    for (int m = 0; m < 10; ++m) { accA[m] = V(T(0)); accB[m] = V(T(0)); }
    __syncthreads();                                  // (aux: halo columns of the first plane)
    int ms = 0;
    for (int i = 0; i < NI; ++i) {
      const int k = kb + i;
      if (i < NG) {
        mbar_wait(&bars[ms], (uint32_t)((i / S) & 1));
        xpass(ms, A0);
      }
      __syncthreads();
      if (t == 0 && i + 2 < NG) issue(i + 2);
      if (i < NG) {
        // y-pull (a+ from the row below, a- from the row above, own a0) and z-push
        V outm[10];
#pragma unroll
        for (int m = 0; m < 10; ++m) outm[m] = accA[m];
        constexpr int MI[3][3][3] = {{{0, 3, 6}, {2, 9, -1}, {5, -1, -1}}, {{1, 8, -1}, {7, -1, -1}, {-1, -1, -1}}, {{4, -1, -1}, {-1, -1, -1}, {-1, -1, -1}}};
#pragma unroll
        for (int p = 0; p < 3; ++p) {
          V Yq[3][3];
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            const V up = lds_pair(s_ap + (3 * c + p) * YPF + oY - TX);
            const V dn = lds_pair(s_am + (3 * c + p) * YPF + oY + TX);
            pull3<V, T>(up, dn, A0[3 * c + p], Yq[0][c], Yq[1][c], Yq[2][c]);
          }
#pragma unroll
          for (int q = 0; q + p <= 2; ++q) {
            V ap, am, a0;
            push3<3, V, T>(Yq[q][0], Yq[q][1], Yq[q][2], ap, am, a0);
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
        // plane k-1 is complete: u_b = m'/rho', Pi^neq' = Pi' - rho' u_b u_b
        const V inv = prcp<T>(outm[0] + V(T(1)));
        const V ux = outm[1] * inv, uy = outm[2] * inv, uz = outm[3] * inv;
        sts_pair(s_fl + oF, ux); sts_pair(s_fl + FLF + oF, uy); sts_pair(s_fl + 2 * FLF + oF, uz);
        sts_pair(s_fl + 3 * FLF + oF, inv);
        const int jj = k - 1;
        if (jj >= z0 && (P.zper || (jj > 0 && jj < L.nz - 1))) {
          V o[7];
          o[0] = outm[0];
          o[1] = outm[4] - outm[1] * ux; o[2] = outm[5] - outm[2] * uy; o[3] = outm[6] - outm[3] * uz;
          o[4] = outm[7] - outm[1] * uy; o[5] = outm[8] - outm[1] * uz; o[6] = outm[9] - outm[2] * uz;
          const long long zo = (long long)jj * L.plane;
          *reinterpret_cast<V *>(P.out.f[F_DRHO] + zo + o00) = o[0];
#pragma unroll
          for (int m = 0; m < 6; ++m) *reinterpret_cast<V *>(P.out.f[F_PXX + m] + zo + o00) = o[1 + m];
          if (edge) {
            store_ghosts(F_DRHO, zo, o[0]);
#pragma unroll
            for (int m = 0; m < 6; ++m) store_ghosts(F_PXX + m, zo, o[1 + m]);
          }
        }
      }
      __syncthreads();
      ms = ms == S - 1 ? 0 : ms + 1;
    }
  } else if (role == 1) {
    // ======================================= phase threads ======================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
    V nA[3], nB[3];           // own n of planes k-2 and k-1
    V gA(T(0)), gB(T(0));     // own |G| of planes k-2 and k-1
    V c_inpl(T(0)), c_upa(T(0)), c_upb(T(0));
#pragma unroll
    for (int m = 0; m < 3; ++m) { nA[m] = V(T(0)); nB[m] = V(T(0)); }
    __syncthreads();
    int ms = 0, ps = 0, ns = 0;
    for (int i = 0; i < NI; ++i) {
      const int k = kb + i;
      if (i < NG) mbar_wait(&bars[ms], (uint32_t)((i / S) & 1));
      const int ms1 = ms == 0 ? S - 1 : ms - 1;
      const int ns1 = ns == 0 ? NR - 1 : ns - 1;
      const int ns2 = ns1 == 0 ? NR - 1 : ns1 - 1;
      const T *phm = phi_at(ps), *phc = phi_at((ps + 1) % SP), *php = phi_at((ps + 2) % SP);
      if (i < NG) {
        // A1: T = S_y S_z phi, U = d_y S_z phi, V = S_y d_z phi of plane k on the region rows
        for (int e = tt; e < RY * (RX / 2); e += W::NFLOW) {
          const int rr = e / (RX / 2), cp = 2 * (e - rr * (RX / 2));
          const int o = (rr + 1) * RX + cp;
          V sz[3], dz[3];
#pragma unroll
          for (int d = 0; d < 3; ++d) {
            const V a = lds_pair(phm + o + (d - 1) * RX), b = lds_pair(phc + o + (d - 1) * RX), c = lds_pair(php + o + (d - 1) * RX);
            sz[d] = pfma(b, w0, (a + c) * w1);
            dz[d] = (c - a) * T(0.5);
          }
          sts_pair(s_tuv + rr * RX + cp, pfma(sz[1], w0, (sz[0] + sz[2]) * w1));
          sts_pair(s_tuv + PL + rr * RX + cp, (sz[2] - sz[0]) * T(0.5));
          sts_pair(s_tuv + 2 * PL + rr * RX + cp, pfma(dz[1], w0, (dz[0] + dz[2]) * w1));
        }
      }
      if (i >= 1) {
        const int j = k - 2;
        const bool fin = (j >= z0);
        // fluxes of plane k-1
        const T *ph = phm + (r + 1) * RX + c0;
        const T *mo = mom_at(ms1) + oM;
        const T *nr = nrm_at(ns1) + oM;
        const V gamv(P.gamma);
        auto qterm = [&](V p, V u, V n) { return p * pfma(pfma(p, V(T(0)) - gamv, gamv), n, u * T(4)); };
        const V pc = lds_pair(ph);
        const V uxc = lds_pair(mo + F_UX * MF);
        const V pn(ph[-1], ph[2]);
        const V qO = qterm(pc, uxc, nB[0]);
        const V qX = qterm(pn, V(mo[F_UX * MF - 1], mo[F_UX * MF + 2]), V(nr[-1], nr[2]));
        V inpl((pn.x + qX.x) + (pc.y - qO.y), (pc.x + qO.x) + (pn.y - qX.y));
        const V phs = lds_pair(ph - RX), phn_ = lds_pair(ph + RX);
        const V qS = qterm(phs, lds_pair(mo + F_UY * MF - RX), lds_pair(nr + PL - RX));
        const V qN = qterm(phn_, lds_pair(mo + F_UY * MF + RX), lds_pair(nr + PL + RX));
        inpl = inpl + ((phs + qS) + (phn_ - qN));
        inpl = pfma(inpl, T(0.125), pc * T(0.25));
        const V qZ = qterm(pc, lds_pair(mo + F_UZ * MF), nB[2]);
        const V up = pc + qZ, down = pc - qZ;
        if (fin) {
          const V phin = pfma(c_upa + down, T(0.125), c_inpl);
          // kappa(j) = -div n from the z-combined normals
          const T *za = s_zc + oM;
          V own(T(0)), nb(T(0));
#pragma unroll
          for (int dy = -1; dy <= 1; ++dy) {
            const T w = dy == 0 ? w0 : w1;
            own = pfma(lds_pair(za + dy * RX), w, own);
            nb = pfma(V(za[dy * RX - 1], za[dy * RX + 2]), w, nb);
          }
          V kap(T(0.5) * (own.y - nb.x), T(0.5) * (nb.y - own.x));
          const T *zb = za + PL;
          const V dO = lds_pair(zb + RX) - lds_pair(zb - RX);
          const V dN = V(zb[RX - 1], zb[RX + 2]) - V(zb[-RX - 1], zb[-RX + 2]);
          kap.x += T(0.5) * (w1 * dN.x + w0 * dO.x + w1 * dO.y);
          kap.y += T(0.5) * (w1 * dO.x + w0 * dO.y + w1 * dN.y);
          const T *zc_ = za + 2 * PL;
          V eO(T(0)), eN(T(0));
#pragma unroll
          for (int dy = -1; dy <= 1; ++dy) {
            const T w = dy == 0 ? w0 : w1;
            eO = pfma(lds_pair(zc_ + dy * RX), w, eO);
            eN = pfma(V(zc_[dy * RX - 1], zc_[dy * RX + 2]), w, eN);
          }
          kap.x += w1 * eN.x + w0 * eO.x + w1 * eO.y;
          kap.y += w1 * eO.x + w0 * eO.y + w1 * eN.y;
          // kick: u' = u_b + sigma kappa G / rho', kappa = -div n, G = n (|G| + eps)
          const V sc = (kap * (gA + V(T(1e-12)))) * lds_pair(s_fl + 3 * FLF + oF) * (-P.sigma);
          if (P.zper || (j > 0 && j < L.nz - 1)) {
            V o[4];
            o[0] = pfma(nA[0], sc, lds_pair(s_fl + oF));
            o[1] = pfma(nA[1], sc, lds_pair(s_fl + FLF + oF));
            o[2] = pfma(nA[2], sc, lds_pair(s_fl + 2 * FLF + oF));
            o[3] = phin;
            const long long zo = (long long)j * L.plane;
#pragma unroll
            for (int m = 0; m < 3; ++m) *reinterpret_cast<V *>(P.out.f[F_UX + m] + zo + o00) = o[m];
            *reinterpret_cast<V *>(P.out.f[F_PHI] + zo + o00) = o[3];
            if (edge) {
#pragma unroll
              for (int m = 0; m < 3; ++m) store_ghosts(F_UX + m, zo, o[m]);
              store_ghosts(F_PHI, zo, o[3]);
            }
          }
        }
        c_upa = c_upb; c_upb = up; c_inpl = inpl;
      }
      __syncthreads();
      if (i < NG) {
        // G = (d_x T, S_x U, S_x V), n = G/(|G|+eps) of plane k on tile+1 -> ring slot ns
        T *nk = nrm_at(ns);
        auto gn_pair = [&](int o, int ol, int orr, V nn[3], V &mag) {
          const V tc = lds_pair(s_tuv + o), uc = lds_pair(s_tuv + PL + o), vc = lds_pair(s_tuv + 2 * PL + o);
          const T tl = s_tuv[ol], tr_ = s_tuv[orr], ul = s_tuv[PL + ol], ur = s_tuv[PL + orr];
          const T vl = s_tuv[2 * PL + ol], vr = s_tuv[2 * PL + orr];
          const V gx(T(0.5) * (tc.y - tl), T(0.5) * (tr_ - tc.x));
          const V gy(w1 * (ul + uc.y) + w0 * uc.x, w1 * (uc.x + ur) + w0 * uc.y);
          const V gz(w1 * (vl + vc.y) + w0 * vc.x, w1 * (vc.x + vr) + w0 * vc.y);
          const V s2 = pfma(gz, gz, pfma(gy, gy, gx * gx));
          mag = V(sqrt1(s2.x), sqrt1(s2.y));
          const V inv(rcp1(mag.x + T(1e-12)), rcp1(mag.y + T(1e-12)));
          nn[0] = gx * inv; nn[1] = gy * inv; nn[2] = gz * inv;
          sts_pair(nk + o, nn[0]); sts_pair(nk + PL + o, nn[1]); sts_pair(nk + 2 * PL + o, nn[2]);
        };
        {
          V nC[3], gC;
          gn_pair(oM, oM - 1, oM + 2, nC, gC);
          sts_pair(s_zc + oM, pfma(nB[0], w0, (nA[0] + nC[0]) * w1));
          sts_pair(s_zc + PL + oM, pfma(nB[1], w0, (nA[1] + nC[1]) * w1));
          sts_pair(s_zc + 2 * PL + oM, (nC[2] - nA[2]) * T(0.5));
#pragma unroll
          for (int a = 0; a < 3; ++a) { nA[a] = nB[a]; nB[a] = nC[a]; }
          gA = gB; gB = gC;
        }
        // ring of tile+1: rows 0 and RY-1 (cols HL-2 .. HL+TX+1) and the two outer column pairs
        constexpr int PPR = TX / 2 + 2;
        constexpr int NT = 2 * PPR + 2 * TY;
        const T *n1 = nrm_at(ns1), *n2 = nrm_at(ns2);
        for (int e = tt; e < NT; e += W::NFLOW) {
          int rr, c;
          if (e < 2 * PPR) { rr = (e < PPR) ? 0 : RY - 1; c = HL - 2 + 2 * (e % PPR); }
          else { const int q = e - 2 * PPR; rr = 1 + (q >> 1); c = (q & 1) ? HL + TX : HL - 2; }
          const int o = rr * RX + c;
          const int ol = c > 0 ? o - 1 : o, orr = c + 2 < RX ? o + 2 : o + 1;
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
      __syncthreads();
      ms = ms == S - 1 ? 0 : ms + 1;
      ps = ps == SP - 1 ? 0 : ps + 1;
      ns = ns == NR - 1 ? 0 : ns + 1;
    }
  } else {
    // ========================================= aux warp =========================================
    // x-pass terms of the halo columns x0-1 (a+) and x0+TX (a-) of every region row of a plane
    auto halo_cols = [&](int slot) {
      const int e = tt;
      if (e < 2 * RY) {
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
    V A0[9];
    mbar_wait(&bars[0], 0u);
    halo_cols(0);
    __syncthreads();
    int ms = 0;
    for (int i = 0; i < NI; ++i) {
      if (i < NG) {
        mbar_wait(&bars[ms], (uint32_t)((i / S) & 1));
        xpass(ms, A0);
      }
      __syncthreads();
      if (i + 1 < NG) {
        const int sl = ms == S - 1 ? 0 : ms + 1;
        mbar_wait(&bars[sl], (uint32_t)(((i + 1) / S) & 1));
        halo_cols(sl);
      }
      __syncthreads();
      ms = ms == S - 1 ? 0 : ms + 1;
    }
  }
}

// host side: launch (fp32, two-component only); the jet boundary planes follow as in launch_tiled_t
template <int TX, int TY>
cudaError_t launch_tiled_ws(TiledPlan &pl, const StepParams<float> &P, int src, int order, cudaStream_t st) {
  using W = WsCfg<TX, TY>;
  const TiledMaps &M = pl.maps[src];
  dim3 grid(M.ntx * M.nty, (P.L.nz + M.zc - 1) / M.zc);
  cudaError_t e = cudaSuccess;
  static bool attr_set = false;
  if (!attr_set) {
    e = cudaFuncSetAttribute(tiled_ws_kernel<TX, TY, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)W::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(tiled_ws_kernel<TX, TY, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)W::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  if (order >= 3) tiled_ws_kernel<TX, TY, 3><<<grid, W::NTHREADS, W::SMEM_BYTES, st>>>(P, M);
  else tiled_ws_kernel<TX, TY, 2><<<grid, W::NTHREADS, W::SMEM_BYTES, st>>>(P, M);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (!P.zper) {
    dim3 b(128), g((P.L.px + 127) / 128, P.L.py, 2);
    tiled_boundary_kernel<float><<<g, b, 0, st>>>(P, 1);
    e = cudaGetLastError();
  }
  return e;
}

}  // namespace tslb
