// tslb_tiled.cuh -- the fused TSLB step as ONE TMA-staged kernel (sm_100a).
//
// Work decomposition.  A CTA owns an x-y tile of TX x TY nodes and MARCHES along z
// over a chunk of planes.  Per plane k it receives, by TMA (cp.async.bulk.tensor, one 4-D box for
// the ten moment arrays and one 3-D box for phi, completion on an mbarrier), the old moments of
// plane k on tile+halo and the old phi of plane k+1 into 3-stage shared-memory rings, prefetched
// three planes ahead.  Every thread owns TWO x-adjacent nodes (packed fp32 math, tslb_pair.cuh).
//
// The 27-neighbour pull of PAPER.md:98 eq. 6 / Fig. 1 is evaluated in the tensor-product Hermite
// basis (tslb_math.cuh) as three 1-D three-point passes:
//   x-pass  K_abc (17 per node, evaluated once) in push form: a+ / a- cross to the neighbouring
//           lane inside the warp -> X^p_bc (24 per node, registers);
//   y-push  every row forms, per (p,c), the combination a+ it sends to the row above, a- it sends
//           to the row below and a0 it keeps: 9+9 values per node cross shared memory, in a
//           double-buffered field that the neighbouring rows read ONE ITERATION LATER -> Y^pq_c;
//   z-push  Y^pq_c of source plane k-1 is pushed into the register accumulators of the destination
//           planes k-2, k-1, k (two live accumulator sets);
// so each stored moment is read from HBM once and the populations never exist in memory.
// The phase-field half (eqs. 20-24) runs in the same kernel from the phi ring.
// Every thread keeps, for its own node pair, the in-plane combinations D_x S_y phi, S_x D_y phi,
// S_x S_y phi of the last three planes in registers, so G = grad(phi) and n = G/(|G|+eps) need nine
// shared-memory loads per plane and no intermediate array; what crosses shared memory are the
// z-combined normals (for kappa = -div n) and the D3Q7 fluxes phi +- q each node sends to its four
// in-plane neighbours (push form) -- phi, grad(phi), n and kappa never touch HBM.
//
// Thread roles: TY/2 "compute" warps own the tile (two rows each); one warp does the x-pass and the
// phase geometry of the two halo rows; 2 RY lanes of a last warp own the two halo columns (their
// x-pass terms one plane ahead, their phase geometry) and its last lane issues the TMA loads.
// Everything a thread reads from another warp was written one iteration earlier into the other half
// of a double buffer: ONE __syncthreads per plane.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <string>
#include <type_traits>

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
  // UNI (fp64, two components): ONE copy of the phase code -- every phase thread owns one
  // node pair, and the pairs of the two halo rows are owned by a phase warp of their own that runs the same
  // code with its stores switched off -- so that the code the SM's warps loop over fits the 32 KB instruction
  // cache; and the flow work of a plane is split between the warps that form the x-pass / y-push terms (A)
  // and the warps that pull them one iteration later, push along z, finish and store the plane (C, D), so
  // that no warp carries more than ~500 instructions per plane.  Register classes by warpgroup (setmaxnreg):
  // warps 0-3 A (three for the tile rows, one for the halo rows), 4-6 C + D and 7 the halo columns, 8-11 phase.
  static constexpr bool UNI = TWO && sizeof(T) == 8;
  static_assert(LX == 16 && TY % (UNI ? 2 : 4) == 0, "a warp owns two rows of 16 node pairs; a phase warp four rows (UNI: two)");
  // left/right staged halo columns.  2 are needed; the TMA box row must be a multiple of 32 bytes
  // (16-byte-odd rows raised "illegal instruction" on B200), so fp32 stages 4.
  static constexpr int HL = sizeof(T) == 4 ? 4 : 2;
  static constexpr int RX = TX + 2 * HL;   // staged columns x0-HL .. x0+TX+HL-1
  static constexpr int RY = TY + 2;        // staged moment rows y0-1 .. y0+TY   ("region rows")
  static constexpr int RYP = TY + 4;       // staged phi rows y0-2 .. y0+TY+1
  static constexpr int S = 3;              // TMA ring depth (group = moments of plane k + phi of plane k+2)
  // warp roles: NWF flow warps (two tile rows each), the halo-row warp, the halo-column warp, and (two-
  // component) NWP phase warps that own the phase field of four tile rows each
  static constexpr int NWF = TY / 2;
  static constexpr int NWP = TWO ? (UNI ? TY / 2 + 1 : TY / 4) : 0;
  static constexpr int W_HALO = NWF, W_C0 = NWF + 1;          // (W_C0: UNI, first of the NWF C warps)
  static constexpr int W_COL = UNI ? W_C0 + NWF : NWF + 1, W_PH0 = UNI ? W_COL + 1 : NWF + 2;
  static_assert(!UNI || (NWF + 1 == 4 && NWP == 4), "UNI: A warps, C warps + halo-column warp, phase warps: a warpgroup each");
  // (setmaxnreg is a warpgroup instruction, and the register pool of the CTA is what its warps were launched with)
  static constexpr int NTHREADS = UNI ? 384 : 32 * (NWF + 2 + NWP);
  static constexpr int NXPASS = 32 * (NWF + 1);          // threads that take part in the x-pass / y-push
  static_assert(2 * RY < 32, "the halo-column warp has one lane per halo-column node and a spare lane");
  static constexpr int NYP = 9;            // y-push fields per direction: (c,p)
  static constexpr int ZW = TX + 4;        // columns x0-2 .. x0+TX+1 of a z-combined-normal array
  static constexpr int FQW = LX + 2;       // node pairs per region row incl. the two halo-column pairs
  static constexpr size_t al(size_t b) { return (b + 127) / 128 * 128; }
  static constexpr size_t MOM_BYTES = (size_t)10 * RY * RX * sizeof(T);   // one TMA box
  static constexpr size_t PHI_BYTES = (size_t)RYP * RX * sizeof(T);
  static constexpr size_t MOM_STAGE = al(MOM_BYTES);
  static constexpr size_t PHI_STAGE = al(PHI_BYTES);
  // Exchange arrays, in ELEMENTS.  Everything that one warp writes and another reads one iteration later
  // lives in a block that exists twice (index = plane parity), all arrays at the same offsets, so that one
  // register (parity x block size) selects the half.
  static constexpr int ZCE = RY * ZW;      // x-combined z-combinations of n: region rows x ZW columns
  static constexpr int ZLE = 2 * RY + 4;   // the same z-combinations, raw, on the two halo columns
  static constexpr int GQE = RY * TX;      // region rows x tile columns
  static constexpr int FQE = RY * FQW;     // one scalar per node pair
  static constexpr int TLE = TY * TX;      // tile nodes
  static constexpr int B_ZC = 0;                                 // [3]  D_x S_z n_x, S_x S_z n_y, S_x d_z n_z
  static constexpr int B_ZL = B_ZC + (TWO ? 3 * ZCE : 0);        // [3]  S_z n_x, S_z n_y, d_z n_z on the halo columns
  static constexpr int B_ZZ = B_ZL + (TWO ? 3 * ZLE : 0);        // [3]  zeros (what the lanes off the tile edge read)
  static constexpr int B_GQ = B_ZZ + (TWO ? 3 * ZLE : 0);        // [2]  phi + q_y, phi - q_y
  static constexpr int B_FQ = B_GQ + (TWO ? 2 * GQE : 0);        // [2]  (phi + q_x).y, (phi - q_x).x per pair
  static constexpr int B_KF = B_FQ + (TWO ? 2 * FQE : 0);        // [3]  F = sigma kappa grad(phi), phase -> flow
  static constexpr int B_PH = B_KF + (TWO && !UNI ? 3 * TLE : 0);   // [1]  own phi, private to the owning phase thread
  static constexpr int PHE = UNI ? GQE : TLE;                    //      (UNI: of the halo-row pairs too)
  static constexpr int BUF = (B_PH + (TWO ? PHE : 0) + 3) / 4 * 4;   // elements per half
  static_assert(ZCE % 2 == 0 && ZLE % 2 == 0 && GQE % 2 == 0 && FQE % 2 == 0, "pair alignment");
  // y-push field: TY sending rows, and one more row that holds the x-pass terms of a halo column for the
  // lanes at the tile edge ([2 plane parities][RY]; a+ of column x0-1 in the a+ fields, a- of column
  // x0+TX in the a- fields), so that they sit at the same field stride as the lanes' own x-exchange words
  static constexpr int YPF = (TY + 1) * TX;
  static_assert(2 * RY <= TX, "halo-column terms fit one row");
  static constexpr size_t OFF_MOM = 0;
  static constexpr size_t OFF_PHI = OFF_MOM + S * MOM_STAGE;
  static constexpr size_t OFF_BUF = OFF_PHI + (TWO ? S * PHI_STAGE : 0);    // [2][BUF]
  // y-push fields: a+ of region rows 0..TY-1 and a- of region rows 2..TY+1 (written and read inside one
  // iteration, between the x-pass barrier and the CTA barrier)
  // grad(phi) of the tile nodes, written by the phase thread that owns the pair and read two iterations
  // later by whoever forms F: a ring of three slots (slot = TMA ring slot of the writing iteration)
  static constexpr size_t OFF_GR = OFF_BUF + (size_t)2 * BUF * sizeof(T);   // [3][3][TLE]
  // (UNI: the y-push fields and the rows' own terms a0 cross an iteration -- A writes, C reads one iteration
  // later -- and exist twice, by plane parity)
  static constexpr int NCOPY = UNI ? 2 : 1;
  static constexpr size_t OFF_AP = OFF_GR + (TWO ? (size_t)9 * TLE * sizeof(T) : 0);   // [NCOPY][9][YPF]
  static constexpr size_t OFF_AM = OFF_AP + (size_t)NCOPY * NYP * YPF * sizeof(T);     // [NCOPY][9][YPF]
  static constexpr size_t OFF_A0 = OFF_AM + (size_t)NCOPY * NYP * YPF * sizeof(T);     // UNI: [2][9][TLE]
  static constexpr size_t OFF_BAR = OFF_A0 + (UNI ? (size_t)2 * NYP * TLE * sizeof(T) : 0);
  static constexpr size_t SMEM_BYTES = OFF_BAR + 64;
  static_assert(SMEM_BYTES <= 227 * 1024, "shared memory of one CTA");
  static constexpr int CTAS_PER_SM = SMEM_BYTES <= 113 * 1024 ? 2 : 1;
};

struct TiledMaps {
  CUtensorMap mom;   // 4-D (px, py, nz, 10) over the SOURCE buffer, box (RX, RY, 1, 10)
  CUtensorMap phi;   // 3-D (px, py, nz) over the source phi, box (RX, RYP, 1)
  int ntx, nty;      // tiles per row / column
  unsigned fsh;      // half the spacing of the field arrays of a buffer, in bytes
  int zc;            // planes per z chunk
};

// Reciprocal and square root.  fp32: the branch-free MUFU approximations (<= 2 ulp, far inside the
// 1e-5 parity gate; rho' ~ 1 and |G| + eps >= 1e-12 are normal numbers).  fp64: the 20-bit MUFU seed and
// two Newton steps (+ a residual step for the root), branch-free: the compiler's IEEE sequences carry an
// out-of-line special-case path that sqrt(0) -- every node away from the interface -- takes, and the
// code has to stay inside the instruction cache.  Within 1 ulp of the IEEE result; a root of less than
// 1e-140 (its square is flushed by the seed) is returned as 0, which moves n = G/(|G| + 1e-12) by < 1e-128.
__device__ __forceinline__ float rcp1(float s) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s)); return r; }
__device__ __forceinline__ double rcp1(double s) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(s));
  r = fma(r, fma(-s, r, 1.0), r);
  return fma(r, fma(-s, r, 1.0), r);
}
__device__ __forceinline__ float sqrt1(float s) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s)); return r; }
__device__ __forceinline__ double sqrt1(double s) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
  double g = s * y, h = 0.5 * y, e = fma(-g, h, 0.5);
  g = fma(g, e, g); h = fma(h, e, h);
  e = fma(-g, h, 0.5);
  g = fma(g, e, g); h = fma(h, e, h);
  g = fma(fma(-g, g, s), h, g);
  return s < 1e-280 ? 0.0 : g;
}
template <typename T> __device__ __forceinline__ Pair<T> prcp(Pair<T> a) { return Pair<T>(rcp1(a.x), rcp1(a.y)); }

// predicated shared-memory pair store (kept as ONE predicated instruction: a branch around a store
// costs a convergence barrier per store in the x-pass)
__device__ __forceinline__ void sts_pair_if(bool p, float *a, Pair<float> v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %0, 0;\n@q st.shared.v2.f32 [%1], {%2, %3};\n}"
               ::"r"((int)p), "r"(smem_u32(a)), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void sts_pair_if(bool p, double *a, Pair<double> v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %0, 0;\n@q st.shared.v2.f64 [%1], {%2, %3};\n}"
               ::"r"((int)p), "r"(smem_u32(a)), "d"(v.x), "d"(v.y) : "memory");
}

// predicated shared-memory load into v (one predicated instruction, no branch)
__device__ __forceinline__ void lds_if(int p, const float *a, float &v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q ld.shared.f32 %0, [%1];\n}" : "+f"(v) : "r"(smem_u32(a)), "r"(p) : "memory");
}
__device__ __forceinline__ void lds_if(int p, const double *a, double &v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q ld.shared.f64 %0, [%1];\n}" : "+d"(v) : "r"(smem_u32(a)), "r"(p) : "memory");
}

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

// Per-node-pair state of the phase-field half that a thread carries from plane to plane in registers.
// At the start of iteration k (the newest phi plane seen is k+1):
template <typename T>
struct PhaseState {
  typedef Pair<T> V;
  V P1b, P2b, P3b;   // D_x S_y phi, S_x D_y phi, S_x S_y phi of plane k+1
  V A1, A2;          // w1 P(k) + w0 P(k+1) of the first two: G(k+1) = A + w1 P(k+2)
  V D3;              // -1/2 P3(k):                             G_z(k+1) = D3 + 1/2 P3(k+2)
  V nB[3];           // n(k)
  V ZA, ZB, DZ;      // w1 n_x(k-1) + w0 n_x(k), the same of n_y, -1/2 n_z(k-1): z-combinations of plane k in the making
  V acc, cup;        // phi'(k-1) in the making: phi/4 + (own cross terms + up(k-2))/8;  up(k-1)
  __device__ __forceinline__ void clear() {
    const V z(T(0));
    P1b = P2b = P3b = A1 = A2 = D3 = ZA = ZB = DZ = acc = cup = z;
#pragma unroll
    for (int a = 0; a < 3; ++a) nB[a] = z;
  }
};

template <int N> using IC = std::integral_constant<int, N>;

// Where a node pair sits in the staged arrays of the CTA: offset of its row r in a staged plane, staged
// column c0 of its first node, the two outer columns (clamped: unused halves), its offsets in the
// z-combined-normal, flux-scalar, tile-column and tile arrays.
struct PairGeom {
  int oP, c0, cl, cr, oZ, oF, oG, oT;
};

// predicated global pair store (one instruction, no branch)
__device__ __forceinline__ void stg_pair_if(bool p, float *a, Pair<float> v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %0, 0;\n@q st.global.cs.v2.f32 [%1], {%2, %3};\n}"
               ::"r"((int)p), "l"(a), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void stg_pair_if(bool p, double *a, Pair<double> v) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %0, 0;\n@q st.global.cs.v2.f64 [%1], {%2, %3};\n}"
               ::"r"((int)p), "l"(a), "d"(v.x), "d"(v.y) : "memory");
}
// Periodic ghost images of a node pair next to the domain edge: element offsets from the pair to its x image
// (dx = +-nx) and its y image (dy = +-ny px), 0 where it has none (hx, hy), and whether the tile of the CTA touches
// the domain edge in x / in y at all (cx, cy: uniform over the CTA -- the tiles inside the domain skip the code, the
// tiles at the edge pay one predicated store per field and image; the rolled loop over the images that stood here
// before cost the edge tiles a third of their instructions, 5 % of the C5 step).
struct ImgGeom {
  bool cx, cy, hx, hy;
  int dx, dy;      // (ny px < 2^31: tiled_supported)
};
template <typename T>
__device__ __forceinline__ T *field_at(T *p0, unsigned fsh, int m) {
  return reinterpret_cast<T *>(reinterpret_cast<char *>(p0) + (unsigned long long)fsh * (unsigned)(2 * m));
}
template <typename T, unsigned MASK>
__device__ __forceinline__ void store_images(const Pair<T> *o, T *p0, unsigned fsh, const ImgGeom &g, bool en) {
  if (g.cx) {
    T *q = p0 + g.dx;
#pragma unroll
    for (int m = 0; m < NF_MAX; ++m)
      if (MASK >> m & 1u) stg_pair_if(en && g.hx, field_at(q, fsh, m), o[m]);
  }
  if (g.cy) {
    T *q = p0 + g.dy;
#pragma unroll
    for (int m = 0; m < NF_MAX; ++m)
      if (MASK >> m & 1u) stg_pair_if(en && g.hy, field_at(q, fsh, m), o[m]);
    if (g.cx) {
      q += g.dx;
#pragma unroll
      for (int m = 0; m < NF_MAX; ++m)
        if (MASK >> m & 1u) stg_pair_if(en && g.hx && g.hy, field_at(q, fsh, m), o[m]);
    }
  }
}

// The rare part of a store of the fields of MASK (bit m = field m) of one node pair of plane j at (gx, gy) on a
// slab face: the same values into the neighbour slab's ghost planes through its peer pointers (phi from the two
// planes next to the face, the moments from the face plane).  (img: also the periodic ghost images in the own
// buffer -- unused since store_images.)
template <typename T, unsigned MASK, bool SLAB>
__device__ __forceinline__ void store_rare(const StepParams<T> &P, const Pair<T> *o, int j, int gx, int gy, bool img) {
  typedef Pair<T> V;
  const Layout &L = P.L;
  const bool push = SLAB && ((j < 2 && P.nb[0].f[0]) || (j >= L.nz - 2 && P.nb[1].f[0]));
  if (img || push) {
    const long long zo = (long long)j * L.plane;
    const int gxg = gx < 2 ? gx + L.nx : (gx >= L.nx - 2 ? gx - L.nx : gx);
    const int gyg = gy < GY ? gy + L.ny : (gy >= L.ny - GY ? gy - L.ny : gy);
    const long long o00 = L.idx(gx, gy, 0), o10 = L.idx(gxg, gy, 0), o01 = L.idx(gx, gyg, 0), o11 = L.idx(gxg, gyg, 0);
    if (img) {
#pragma unroll 1
      for (int im = 0; im < 3; ++im) {       // one copy of the store code: x image, y image, corner
        if (im == 0 ? gxg == gx : (im == 1 ? gyg == gy : (gxg == gx || gyg == gy))) continue;
        const long long og = zo + (im == 0 ? o10 : (im == 1 ? o01 : o11));
#pragma unroll
        for (int m = 0; m < NF_MAX; ++m)
          if (MASK >> m & 1u) *reinterpret_cast<V *>(P.out.f[m] + og) = o[m];
      }
    }
    if (push) {
#pragma unroll 1
      for (int side = 0; side < 2; ++side) {
        const int depth = side == 0 ? j : L.nz - 1 - j;
        if (!P.nb[side].f[0] || depth > 1) continue;
        const long long zn = (long long)(j + P.nb_dz[side]) * L.plane;
#pragma unroll 1
        for (int im = 0; im < 4; ++im) {     // the node itself, then its x / y / corner images
          if (im == 1 ? gxg == gx : (im == 2 ? gyg == gy : (im == 3 && (gxg == gx || gyg == gy)))) continue;
          const long long og = zn + (im == 0 ? o00 : (im == 1 ? o10 : (im == 2 ? o01 : o11)));
#pragma unroll
          for (int m = 0; m < NF_MAX; ++m)
            if ((MASK >> m & 1u) && (depth == 0 || m == F_PHI)) *reinterpret_cast<V *>(P.nb[side].f[m] + og) = o[m];
        }
      }
    }
  }
}
// streaming global pair store (st.global.cs: the new moments are not read again in this step, and should not push the
// old moments that a neighbouring tile is about to read out of L2)
__device__ __forceinline__ void stg_stream(float *a, Pair<float> v) {
  asm volatile("st.global.cs.v2.f32 [%0], {%1, %2};" ::"l"(a), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void stg_stream(double *a, Pair<double> v) {
  asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(a), "d"(v.x), "d"(v.y) : "memory");
}
// Store the fields of MASK (bit m = field m) of one node pair of plane j.  p0: field 0 at this pair and
// plane; the field arrays of a buffer are equally spaced (fsh = half the spacing in bytes, 32 bits: the address
// of field m is then ONE multiply-add, IMAD.WIDE.U32).
template <typename T, unsigned MASK, bool SLAB>
__device__ __forceinline__ void store_pair(const StepParams<T> &P, const Pair<T> *o, T *p0, int j, int gx, int gy,
                                           const ImgGeom &img, unsigned fsh) {
#pragma unroll
  for (int m = 0; m < NF_MAX; ++m)
    if (MASK >> m & 1u) stg_stream(field_at(p0, fsh, m), o[m]);
  store_images<T, MASK>(o, p0, fsh, img, true);
  if (SLAB) store_rare<T, MASK, SLAB>(P, o, j, gx, gy, false);
}
constexpr unsigned FM_U = 0xEu, FM_RHOPI = 0x3F1u, FM_FLOW = 0x3FFu, FM_PHI = 0x400u;   // field masks

// ------------------------------------------------------------------ the kernel
// SLAB: the context is a z-slab (halo faces, ghost planes, halo push).  A separate instantiation
// keeps the single-GPU kernel's loop body small (instruction cache).
//
// Schedule.  Iteration k (k = z0-4 .. z1+1 for the chunk [z0, z1)) ends with the ONE CTA barrier:
//   flow warps   A  K, x-pass and y-push terms of plane k (+ the halo-row warp for the two halo rows);
//                   a barrier among these five warps only;
//                C  y-pull of plane k, z-push: the flow moments of plane k-1 are complete; store rho' and
//                   Pi^neq' of plane k-1; kick u'(k-2) = u_b(k-2) + F(k-2)/rho' with the F the phase warps
//                   wrote in iteration k-1; store u' of plane k-2;
//   halo-col warp   x-pass terms of the two halo columns of plane k+1 (one iteration ahead); B for the
//                   halo-column pairs and the halo-row pairs; its spare lane issues the TMA group of plane
//                   k+3 after the barrier;
//   phase warps  D  kappa(k-1) from the x-combined z-combinations of n written in iteration k-1;
//                   F(k-1) = sigma kappa grad(phi) -> flow warps;
//                B  P(k+2) from the phi ring, G(k+1), n(k+1); z-combinations of n of plane k, combined
//                   along x; fluxes phi +- q of plane k; phi'(k-1), stored at once.
// Everything a warp reads from another role was written one iteration earlier into the other half of
// the double-buffered exchange block.  The iterations before z0-1 only run B (they start the three-plane
// history of the phase geometry).
template <typename T, int TX, int TY, int ORDER, bool TWO, bool SLAB>
__global__ void __launch_bounds__(TileCfg<T, TX, TY, TWO>::NTHREADS, TileCfg<T, TX, TY, TWO>::CTAS_PER_SM)
tiled_step_kernel(const __grid_constant__ StepParams<T> P, const __grid_constant__ TiledMaps M) {
  using C = TileCfg<T, TX, TY, TWO>;
  using V = Pair<T>;
  constexpr int LX = C::LX, HL = C::HL, RX = C::RX, RY = C::RY, S = C::S, ZW = C::ZW, FQW = C::FQW;
  constexpr int ZCE = C::ZCE, ZLE = C::ZLE, GQE = C::GQE, FQE = C::FQE, TLE = C::TLE, YPF = C::YPF, BUF = C::BUF;
  constexpr int MF = RY * RX;                           // elements per moment field in a stage
  constexpr bool UNI = C::UNI;
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::OFF_BAR);
  auto mom_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_MOM + slot * C::MOM_STAGE); };
  auto phi_at = [&](int slot) { return reinterpret_cast<T *>(smem + C::OFF_PHI + slot * C::PHI_STAGE); };
  T *s_buf = reinterpret_cast<T *>(smem + C::OFF_BUF);     // [2][BUF]
  T *s_gr = reinterpret_cast<T *>(smem + C::OFF_GR);       // [3][3][TLE]
  T *s_ap = reinterpret_cast<T *>(smem + C::OFF_AP);       // [9][YPF]  (UNI: [2][9][YPF], by plane parity)
  T *s_am = reinterpret_cast<T *>(smem + C::OFF_AM);
  T *s_a0 = reinterpret_cast<T *>(smem + C::OFF_A0);       // UNI: [2][9][TLE]

  const Layout &L = P.L;
  const int t = threadIdx.x;
  const int lane = t & 31, wid = t >> 5;
  const bool flow = wid < C::NWF;                         // owns the flow of two tile rows
  const bool halow = wid == C::W_HALO;
  const bool colw = wid == C::W_COL;
  const bool phalo = UNI && wid == C::W_PH0 + C::NWP - 1;   // UNI: the phase warp of the two halo rows
  const bool cwarp = UNI && wid >= C::W_C0 && wid < C::W_COL;   // UNI: the warps that run C and D (tile rows like the A warps)
  const int lx = lane & (LX - 1), hi = lane >> 4;
  // region row (y = y0 - 1 + r) of the thread's (first) node pair and staged column of its first node
  const int r = flow ? 2 * wid + 1 + hi
                     : (halow ? (hi ? 0 : RY - 1)
                              : (colw ? (lane < RY ? lane : (lane < 2 * RY ? lane - RY : 0))
                                      : (UNI ? (phalo ? (hi ? 0 : RY - 1) : 2 * (wid - (cwarp ? C::W_C0 : C::W_PH0)) + 1 + hi)
                                             : 4 * (wid - C::W_PH0) + 1 + hi)));
  const int cside = lane >= RY;                           // halo-column warp: 0 left, 1 right
  const int c0 = colw ? (cside ? HL + TX : HL - 2) : HL + 2 * lx;
  int oM = r * RX + c0;                                   // offset of the pair in a staged region plane
  int oT = (r - 1) * TX + 2 * lx;                         // ... in an array over the tile
  // Tile origin.  When nx (ny) is not a multiple of the tile, the last tile of the row (column) is
  // shifted back to end at the domain edge; it recomputes the overlap but stores only its own nodes.
  const int xs = (blockIdx.x % M.ntx) * TX, ys = (blockIdx.x / M.ntx) * TY;
  const int x0 = min(xs, L.nx - TX), y0 = min(ys, L.ny - TY);
  const int z0 = blockIdx.y * M.zc;
  const int z1 = min(z0 + M.zc, L.nz);
  // first iteration's plane: two-component chunks start the three-plane history of the phase geometry
  // at z0-4; single-component chunks need one iteration for the halo columns before the first x-pass
  const int kst = TWO ? z0 - 4 : z0 - 2;
  const int kfirst = TWO ? kst : z0 - 1; // first plane that has a TMA group
  const int NI = z1 - kst + 2;           // iterations: k = kst .. z1+1
  // The same in iteration numbers i = k - kst (what the loops test: no plane arithmetic per iteration):
  // plane z0 is iteration I0, plane z1 iteration IZ1.
  constexpr int I0 = TWO ? 4 : 2;
  const int IZ1 = I0 + (z1 - z0);

  // plane coordinate in the tensor map: wrapped / clamped / ghost plane of a slab (zsrc), shifted
  // by the ghost planes below z = 0
  auto zmap = [&](int z) { return zsrc(P, z) + L.gz; };
  // group of plane k: moments of plane k (source planes z0-1 .. z1) and phi of plane k+2 (planes
  // z0-2 .. z1+1)
  auto has_group = [&](int k) { return k <= z1 && k >= kfirst; };
  auto issue = [&](int k, int slot) {
    uint64_t *bar = &bars[slot];
    const bool mom = k >= z0 - 1, phi = TWO && k < z1;
    mbar_expect_tx(bar, (mom ? (uint32_t)C::MOM_BYTES : 0u) + (phi ? (uint32_t)C::PHI_BYTES : 0u));
    if (mom) tma_load_4d(mom_at(slot), &M.mom, bar, x0 - HL + GX, y0 - 1 + GY, zmap(k), 0);
    if (phi) tma_load_3d(phi_at(slot), &M.phi, bar, x0 - HL + GX, y0 - 2 + GY, zmap(k + 2));
  };

  const bool issuer = t == 32 * C::W_COL + 31;           // spare lane of the halo-column warp
  if (issuer) {
    for (int s = 0; s < S; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (int s = 0; s < S; ++s)
      if (has_group(kfirst + s)) issue(kfirst + s, s);
  }
  if (TWO)   // the zero arrays that the lanes off the tile edge read in D
    for (int e = t; e < 2 * 3 * ZLE; e += C::NTHREADS) s_buf[(e / (3 * ZLE)) * BUF + C::B_ZZ + e % (3 * ZLE)] = T(0);
  __syncthreads();

  const V omc(P.omc);
  const T w1 = T(1.0 / 6.0), w0 = T(2.0 / 3.0);
  const unsigned fs = M.fsh;                             // field arrays are equally spaced: half the spacing in bytes

  // global coordinates / store offset (plane 0) of the thread's (first) pair
  const int gx_ = x0 + 2 * lx, gy_ = y0 + r - 1;
  const long long o00 = L.idx(gx_, gy_, 0);
  // the pair (and, for a phase thread, its second pair two rows up) has a periodic ghost image
  auto img_of = [&](int gx, int gy) {
    ImgGeom g;
    g.cx = x0 < 2 || x0 + TX > L.nx - 2;
    g.cy = y0 < GY || y0 + TY > L.ny - GY;
    g.dx = gx < 2 ? L.nx : (gx >= L.nx - 2 ? -L.nx : 0);
    g.dy = gy < GY ? L.ny * L.px : (gy >= L.ny - GY ? -L.ny * L.px : 0);
    g.hx = g.dx != 0;
    g.hy = g.dy != 0;
    return g;
  };
  const ImgGeom img0 = img_of(gx_, gy_), img1 = img_of(gx_, gy_ + 2);

  // B: phase geometry and fluxes of one node pair (eqs. 20-24, readings A6-A8), iteration k.
  // ROLE 0: a tile pair (finishes and stores phi'); 1: a halo-row pair; 2: a halo-column pair.
  // bo / bn: element offsets of the exchange-block halves of plane parity k&1 / (k-1)&1.
  auto phase_B = [&](auto role, auto drc, PhaseState<T> &st, const PairGeom &g0, int s, int bo, int bn) {
    constexpr int ROLE = decltype(role)::value, DR = decltype(drc)::value;   // DR: rows below the thread's first pair
    const PairGeom g = {g0.oP + DR * RX, g0.c0, g0.cl, g0.cr, g0.oZ + DR * ZW, g0.oF + DR * FQW, g0.oG + DR * TX, g0.oT + DR * TX};
    // in-plane combinations of phi(k+2) on rows r-1, r, r+1 (phi box rows r .. r+2): first along y on the
    // own columns (c) and on the two outer columns (n = (c0-1, c0+2)), then along x
    const T *pp = phi_at(s) + g.oP;
    const V ca = lds_pair(pp + g.c0), cb = lds_pair(pp + RX + g.c0), cc = lds_pair(pp + 2 * RX + g.c0);
    const V na(pp[g.cl], pp[g.cr]), nb(pp[RX + g.cl], pp[RX + g.cr]), nc(pp[2 * RX + g.cl], pp[2 * RX + g.cr]);
    const V syc = pfma(cb, w0, (ca + cc) * w1), dyc = cc - ca;          // S_y phi, 2 D_y phi
    const V syn = pfma(nb, w0, (na + nc) * w1), dyn = nc - na;
    const V sws(syc.y, syc.x), swd(dyc.y, dyc.x);
    const V P1n = (sws - syn) * V(T(0.5), T(-0.5));                     // D_x S_y phi(k+2)
    const V P3n = pfma(syc, w0, (syn + sws) * w1);                      // S_x S_y phi(k+2)
    const V P2n = pfma(dyc, T(1.0 / 3.0), (dyn + swd) * T(1.0 / 12.0)); // S_x D_y phi(k+2)
    // G(k+1) = (S_z P1, S_z P2, D_z P3), n(k+1) = G/(|G| + eps)
    const V gx = pfma(P1n, w1, st.A1), gy = pfma(P2n, w1, st.A2), gz = pfma(P3n, T(0.5), st.D3);
    st.A1 = pfma(P1n, w0, st.P1b * w1); st.P1b = P1n;
    st.A2 = pfma(P2n, w0, st.P2b * w1); st.P2b = P2n;
    st.D3 = st.P3b * T(-0.5); st.P3b = P3n;
    const V s2 = pfma(gz, gz, pfma(gy, gy, gx * gx));
    const V gC(sqrt1(s2.x), sqrt1(s2.y));                               // |G|
    const V ginv(rcp1(gC.x + T(1e-12)), rcp1(gC.y + T(1e-12)));         // reading A7
    const V nCx = gx * ginv, nCy = gy * ginv, nCz = gz * ginv;
    // z-combinations of n of plane k: a = S_z n_x, b = S_z n_y, c = d_z n_z ...
    const V za = pfma(nCx, w1, st.ZA), zb = pfma(nCy, w1, st.ZB), zc = pfma(nCz, T(0.5), st.DZ);
    if (ROLE == 2) {
      // ... of the halo column itself (x0-1: second node of its pair; x0+TX: first node), raw
      T *zl = s_buf + bo + C::B_ZL + cside * RY + 2 + r;
      zl[0] = cside ? za.x : za.y; zl[ZLE] = cside ? zb.x : zb.y; zl[2 * ZLE] = cside ? zc.x : zc.y;
    } else {
      // ... combined along x for kappa(k) = -(D_x S_y a + S_x D_y b + S_x S_y c): the outer columns come
      // from the neighbour lanes; the lanes at the tile edge take 0 (D adds the halo column's share)
      auto outer = [&](V v) {
        const T l = __shfl_up_sync(0xffffffffu, v.y, 1, LX), q = __shfl_down_sync(0xffffffffu, v.x, 1, LX);
        return V(lx == 0 ? T(0) : l, lx == LX - 1 ? T(0) : q);
      };
      const V oa = outer(za), ob = outer(zb), oc = outer(zc);
      T *zw = s_buf + bo + C::B_ZC + g.oZ;
      sts_pair(zw, (V(za.y, za.x) - oa) * V(T(0.5), T(-0.5)));          // D_x a
      sts_pair(zw + ZCE, pfma(zb, w0, (ob + V(zb.y, zb.x)) * w1));      // S_x b
      sts_pair(zw + 2 * ZCE, pfma(zc, w0, (oc + V(zc.y, zc.x)) * w1));  // S_x c
    }
    // a7 in push form: the node sends phi + q_a along +e_a and phi - q_a along -e_a,
    // q_a = phi (4 u_a + gamma (1 - phi) n_a), of plane k
    const T *mo = mom_at(s) + g.oP + g.c0;
    V phinew(T(0));                                                     // phi'(k-1) (tile pairs)
    V ph;                                                               // own phi(k)
    if (ROLE == 0) {
      // tile pairs keep their own phi(k), phi(k+1) in a private two-slot ring (slot = plane parity)
      T *pr = s_buf + bo + C::B_PH + (UNI ? g.oG : g.oT);
      ph = lds_pair(pr);
      sts_pair(pr, cb);
    } else {
      ph = st.acc; st.acc = st.cup; st.cup = cb;                        // (their acc / cup carry phi(k), phi(k+1))
    }
    const V a4 = ph * T(4);
    const V bq = ph * pfma(ph, V(T(0)) - V(P.gamma), V(P.gamma));
    const V qx = pfma(bq, st.nB[0], a4 * lds_pair(mo + F_UX * MF));
    const V qy = pfma(bq, st.nB[1], a4 * lds_pair(mo + F_UY * MF));
    st.ZA = pfma(nCx, w0, st.nB[0] * w1); st.nB[0] = nCx;
    st.ZB = pfma(nCy, w0, st.nB[1] * w1); st.nB[1] = nCy;
    const V fp = ph + qx, fm = ph - qx;
    T *fq = s_buf + bo + C::B_FQ + g.oF;
    fq[0] = fp.y; fq[FQE] = fm.x;
    if (ROLE != 2) {
      T *gq = s_buf + bo + C::B_GQ + g.oG;
      sts_pair(gq, ph + qy);
      sts_pair(gq + GQE, ph - qy);
    }
    if (ROLE == 0) {
      const V qz = pfma(bq, st.nB[2], a4 * lds_pair(mo + F_UZ * MF));
      // grad(phi) of plane k+1 for the kick two iterations on -> ring slot s
      T *gr_ = s_gr + s * 3 * TLE + g.oT;
      if (UNI) { sts_pair_if(!phalo, gr_, gx); sts_pair_if(!phalo, gr_ + TLE, gy); sts_pair_if(!phalo, gr_ + 2 * TLE, gz); }
      else { sts_pair(gr_, gx); sts_pair(gr_ + TLE, gy); sts_pair(gr_ + 2 * TLE, gz); }
      // phi'(k-1) = phi/4 + (in-plane arrivals of plane k-1 + up(k-2) + down(k)) / 8
      const T *fr = s_buf + bn + C::B_FQ + g.oF;
      const T *gr = s_buf + bn + C::B_GQ + g.oG;
      const V xin(fr[-1], fr[FQE + 1]);
      const V yin = lds_pair(gr - TX) + lds_pair(gr + GQE + TX);
      phinew = pfma((xin + yin) + (ph - qz), T(0.125), st.acc);
      st.acc = pfma(V(fm.y, fp.x) + st.cup, T(0.125), ph * T(0.25));
      st.cup = ph + qz;
    }
    st.DZ = st.nB[2] * T(-0.5); st.nB[2] = nCz;
    return phinew;
  };

  // D (run for half of the tile pairs by the phase warp that owns them, for the other half by the halo-row
  // warp, which has time to spare): kappa(k-1) = -(S_y ax + D_y bx + S_y cx) from the x-combined
  // z-combinations of n written in iteration k-1, plus the share of the halo column for the lanes at the tile edge (every other lane reads zeros
  // through the same per-lane pointer: no divergence); F(k-1) = sigma kappa grad(phi)(k-1) -> flow warps.
  // (UNI: the C warp that runs D keeps F in registers, Fr, for its own kick one iteration later)
  auto phase_D = [&](auto drc, int oZ0, int oT0, int s, int bn, int eoff, V emask, T esign, V *Fr) {
    constexpr int DR = decltype(drc)::value;
    const PairGeom g = {0, 0, 0, 0, oZ0 + DR * ZW, 0, 0, oT0 + DR * TX};
    const T *zr = s_buf + bn + C::B_ZC + g.oZ;
    V kap = pfma(lds_pair(zr), w0, (lds_pair(zr - ZW) + lds_pair(zr + ZW)) * w1);                       // S_y D_x a
    kap = pfma(lds_pair(zr + ZCE + ZW) - lds_pair(zr + ZCE - ZW), T(0.5), kap);                         // D_y S_x b
    kap = pfma(lds_pair(zr + 2 * ZCE), w0, pfma(lds_pair(zr + 2 * ZCE - ZW) + lds_pair(zr + 2 * ZCE + ZW), w1, kap));
    const T *ze = s_buf + bn + eoff + DR;
    const T ea = w0 * ze[0] + w1 * (ze[-1] + ze[1]);                     // S_y a on the halo column
    const T eb = ze[ZLE + 1] - ze[ZLE - 1];                              // 2 D_y b
    const T ec = w0 * ze[2 * ZLE] + w1 * (ze[2 * ZLE - 1] + ze[2 * ZLE + 1]);
    const T corr = esign * ea + T(1.0 / 12.0) * eb + w1 * ec;            // -+ a/2 (D_x), w1 b and w1 c (S_x)
    kap = pfma(V(corr), emask, kap);
    const V sc = kap * (-P.sigma);                                       // F = sigma kappa G, kappa = -kap
    const T *gr_ = s_gr + (s == S - 1 ? 0 : s + 1) * 3 * TLE + g.oT;      // G(k-1): written two iterations ago
    if (UNI) {
      Fr[0] = lds_pair(gr_) * sc; Fr[1] = lds_pair(gr_ + TLE) * sc; Fr[2] = lds_pair(gr_ + 2 * TLE) * sc;
    } else {
      T *kf = s_buf + bn + C::B_KF + g.oT;
      sts_pair(kf, lds_pair(gr_) * sc);
      sts_pair(kf + TLE, lds_pair(gr_ + TLE) * sc);
      sts_pair(kf + 2 * TLE, lds_pair(gr_ + 2 * TLE) * sc);
    }
  };

  // ring slot of this iteration's group (group kfirst sits in slot 0) and its mbarrier phase parity
  int s = TWO ? 0 : S - 1;
  uint32_t mph = TWO ? 0u : 1u;
  // end of an iteration: the ONE CTA barrier; in the halo-column warp (ISSUE) the group three planes ahead
  // goes into the slot just read
  auto iter_end = [&](auto issues, int i) {
    __syncthreads();
    if (decltype(issues)::value && issuer && i >= I0 - (TWO ? 4 : 1) && i + S <= IZ1) issue(kst + i + S, s);
    s = s == S - 1 ? 0 : s + 1;
    if (s == 0) mph ^= 1u;
  };

  // A: x-pass of region row r of plane k in push form, then the y-push terms (flow warps and the halo-row
  // warp).  Each node's K is evaluated once; a+ / a- cross to the x-neighbour thread by shuffle (through shared
  // memory the store -> __syncwarp -> load chain sat on the critical path: +1.8 % in fp32); the lanes at the
  // tile edge load the halo column's term instead, which the halo-column warp left in the extra row of the
  // y-push fields one iteration earlier.
  const bool st_ap = r <= TY - 1, st_am = r >= 2;        // rows 0..TY-1 send an a+, rows 2..TY+1 an a-
  // y-push fields: a+ is stored at row index r, a- at r-2; a tile row r reads both at index r-1 (= oT)
  int oAP = r * TX + 2 * lx;
  // the word a lane at the tile edge loads: the halo-column term of row r in the extra row of the y-push
  // fields 0..7 of copy 0 (+ RY for planes of odd parity)
  int oPL = TY * TX + r;
  const int hpar = (lx == 0 ? 1 : 0) | (lx == LX - 1 ? 2 : 0);
  auto xpass = [&](bool odd, int s, V (&A0)[9]) {      // odd: parity of the plane
    const int oAM = oAP - 2 * TX;
    const int yoff = UNI && odd ? C::NYP * YPF : 0;    // UNI: the copy of the y-push fields of this parity
    const T *pl = s_ap + oPL + (odd ? RY : 0), *pr = s_am + oPL + (odd ? RY : 0);
    V Xg[8][3];   // [group][p]
    {
      V m[10], K[NK];
      const T *p = mom_at(s) + oM;
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
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        T l = __shfl_up_sync(0xffffffffu, gp[g].y, 1, LX), q = __shfl_down_sync(0xffffffffu, gm[g].x, 1, LX);
        lds_if(hpar & 1, pl + g * YPF, l);
        lds_if(hpar & 2, pr + g * YPF, q);
        pull3s<V, T>(l, gp[g].x, gm[g].y, q, g0[g], Xg[g][0], Xg[g][1], Xg[g][2]);
      }
    }
    // y-push per (c, p): groups of c = 0: b = 0,1,2 -> g 0,1,2; c = 1: g 3,4,5; c = 2: b = 0,1 -> g 6,7
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int p = 0; p < 3; ++p) {
        V ap, am;
        if (c < 2) push3<3, V, T>(Xg[3 * c][p], Xg[3 * c + 1][p], Xg[3 * c + 2][p], ap, am, A0[3 * c + p]);
        else push3<2, V, T>(Xg[6][p], Xg[7][p], Xg[7][p], ap, am, A0[6 + p]);
        sts_pair_if(st_ap, s_ap + (3 * c + p) * YPF + oAP + yoff, ap);
        sts_pair_if(st_am, s_am + (3 * c + p) * YPF + oAM + yoff, am);
      }
  };
  // the y-push terms of a plane are complete: a barrier among the flow warps and the halo-row warp only
  auto xpass_barrier = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(C::NXPASS) : "memory"); };

  // C: finish the y-pass of a source plane (a+ from the row below, a- from the row above, the rows' own a0)
  // and z-push: am completes the plane below the source plane (-> outm), a0 / ap go on into the accumulators
  auto cstage = [&](const T *yu, const T *yd, auto a0at, V (&accA)[10], V (&accB)[10], V (&outm)[10]) {
    // moment index of (p,q,rr)
    constexpr int MI[3][3][3] = {{{0, 3, 6}, {2, 9, -1}, {5, -1, -1}}, {{1, 8, -1}, {7, -1, -1}, {-1, -1, -1}}, {{4, -1, -1}, {-1, -1, -1}, {-1, -1, -1}}};
#pragma unroll
    for (int p = 0; p < 3; ++p) {
      V Yq[3][3];   // [q][c]
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const V up = lds_pair(yu + (3 * c + p) * YPF);
        const V dn = lds_pair(yd + (3 * c + p) * YPF);
        pull3<V, T>(up, dn, a0at(3 * c + p), Yq[0][c], Yq[1][c], Yq[2][c]);
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
  };

  if (UNI && (flow || halow)) {
    // ============================ UNI: A warps (x-pass and y-push terms of the eight region rows) ============================
    bool odd = kst & 1;                      // parity of plane k: the copy of the y-push fields it goes to
    for (int i = 0; i < NI; ++i) {
      asm volatile("" : "+r"(oM), "+r"(oT), "+r"(oAP), "+r"(oPL));
      if (i <= IZ1) mbar_wait(&bars[s], mph);
      if (i >= I0 - 1 && i <= IZ1) {         // plane k is a source plane of this chunk
        V A0[9];
        xpass(odd, s, A0);
        if (flow) {                          // the tile rows' own terms -> the C warps
          T *a0 = s_a0 + (odd ? C::NYP * TLE : 0) + oT;
#pragma unroll
          for (int q = 0; q < 9; ++q) sts_pair(a0 + q * TLE, A0[q]);
        }
      }
      odd = !odd;
      iter_end(IC<0>(), i);
    }
  } else if (flow || halow) {
    // ============================ flow warps and the halo-row warp ============================
    V accA[10], accB[10];     // Hermite moments being accumulated for planes k and k+1
    V ubx(T(0)), uby(T(0)), ubz(T(0)), rinv(T(1));   // u_b and 1/rho' of the plane completed last
#pragma unroll
    for (int m = 0; m < 10; ++m) { accA[m] = V(T(0)); accB[m] = V(T(0)); }
    // planes this thread stores: its chunk, without the imposed inflow / outflow planes; nothing when the
    // node belongs to the neighbouring (shifted-back) tile
    const int jlo = max(z0, P.jet_lo ? 1 : 0);
    const int njs = (gx_ >= xs && gy_ >= ys) ? min(z1, P.out_hi ? L.nz - 1 : L.nz) - jlo : 0;
    T *pst = P.out.f[0] + o00 + (long long)(kst - 2) * L.plane;   // field 0 of the pair, plane k-2
    const int ju = kst - 2 - jlo;            // (plane k-2) - jlo = i + ju
    bool odd = kst & 1;                      // parity of plane k; bo: its half of the exchange block
    // halo-row warp: D for the second pair of every phase thread (tile rows 3 + hi and 7 + hi)
    const int dZ = (3 + hi) * ZW + 2 + 2 * lx, dT = (2 + hi) * TX + 2 * lx;
    const int deoff = (lx == 0 ? C::B_ZL : (lx == LX - 1 ? C::B_ZL + RY : C::B_ZZ)) + 2 + 3 + hi;
    const V demask(lx == 0 ? T(1) : T(0), lx == LX - 1 ? T(1) : T(0));
    const T design = lx == 0 ? T(-0.5) : T(0.5);
    for (int i = 0; i < NI; ++i) {
      // (keep the loop-invariant offsets in registers: recomputing them from the thread index costs more)
      asm volatile("" : "+r"(oM), "+r"(oT), "+r"(oAP), "+r"(oPL));
      const int bo = odd ? BUF : 0;
      if (i >= (TWO ? 0 : 1) && i <= IZ1) mbar_wait(&bars[s], mph);
      if (TWO && flow && (unsigned)(i + ju) < (unsigned)njs) {
        // a6: u'(k-2) = u_b + F / rho' with the F(k-2) the phase warps wrote in iteration k-1; a9: store it.
        // (First thing in the iteration: u_b and 1/rho' die before the x-pass, and the loads overlap its own.)
        V o[NF_MAX];
        const T *kf = s_buf + bo + C::B_KF + oT;
        o[1] = pfma(lds_pair(kf), rinv, ubx);
        o[2] = pfma(lds_pair(kf + TLE), rinv, uby);
        o[3] = pfma(lds_pair(kf + 2 * TLE), rinv, ubz);
        store_pair<T, FM_U, SLAB>(P, o, pst, kst + i - 2, gx_, gy_, img0, fs);
      }
      const bool src = i >= I0 - 1 && i <= IZ1;    // plane k is a source plane of this chunk
      V A0[9];                               // own y-push term a0 per (c,p)
      if (src) xpass(odd, s, A0);
      xpass_barrier();
      if (TWO && !UNI && halow && i <= IZ1 && i >= I0 + 1) {
        phase_D(IC<0>(), dZ, dT, s, BUF - bo, deoff, demask, design, nullptr);
        phase_D(IC<4>(), dZ, dT, s, BUF - bo, deoff, demask, design, nullptr);
      }
      V o[NF_MAX];
      if (flow && src) {
        // C of plane k: plane k-1 is complete
        V outm[10];
        cstage(s_ap + oT, s_am + oT, [&](int q) { return A0[q]; }, accA, accB, outm);
        // a4: plane k-1 is complete: u_b = m'/rho', Pi^neq' = Pi' - rho' u_b u_b (Hermite form)
        rinv = prcp<T>(outm[0] + V(T(1)));
        ubx = outm[1] * rinv; uby = outm[2] * rinv; ubz = outm[3] * rinv;
        if ((unsigned)(i + ju + 1) < (unsigned)njs) {
          o[0] = outm[0];
          o[4] = outm[4] - outm[1] * ubx;
          o[5] = outm[5] - outm[2] * uby;
          o[6] = outm[6] - outm[3] * ubz;
          o[7] = outm[7] - outm[1] * uby;
          o[8] = outm[8] - outm[1] * ubz;
          o[9] = outm[9] - outm[2] * ubz;
          if (TWO) {
            store_pair<T, FM_RHOPI, SLAB>(P, o, pst + L.plane, kst + i - 1, gx_, gy_, img0, fs);
          } else {
            o[1] = ubx; o[2] = uby; o[3] = ubz;
            store_pair<T, FM_FLOW, SLAB>(P, o, pst + L.plane, kst + i - 1, gx_, gy_, img0, fs);
          }
        }
      }
      pst += L.plane;
      odd = !odd;
      iter_end(IC<0>(), i);
    }
  } else if (colw || cwarp) {
    if (UNI) asm volatile("setmaxnreg.inc.sync.aligned.u32 200;");
    if (cwarp) {
      // ============================ UNI: C warps ============================
      // iteration k: C of source plane k-1 (terms the A warps left in iteration k-1): plane k-2 is complete
      // and, with the F(k-2) formed in iteration k-1, finished and stored; then D: kappa, F of plane k-1
      V accA[10], accB[10], Fr[3];
#pragma unroll
      for (int m = 0; m < 10; ++m) { accA[m] = V(T(0)); accB[m] = V(T(0)); }
      Fr[0] = Fr[1] = Fr[2] = V(T(0));
      const int jlo = max(z0, P.jet_lo ? 1 : 0);
      const int njs = (gx_ >= xs && gy_ >= ys) ? min(z1, P.out_hi ? L.nz - 1 : L.nz) - jlo : 0;
      T *pst = P.out.f[0] + o00 + (long long)(kst - 2) * L.plane;   // field 0 of the pair, plane k-2
      const int ju = kst - 2 - jlo;            // (plane k-2) - jlo = i + ju
      const int oZ = r * ZW + 2 + 2 * lx;
      const int eoff = (lx == 0 ? C::B_ZL : (lx == LX - 1 ? C::B_ZL + RY : C::B_ZZ)) + 2 + r;
      const V emask(lx == 0 ? T(1) : T(0), lx == LX - 1 ? T(1) : T(0));
      const T esign = lx == 0 ? T(-0.5) : T(0.5);
      bool odd = kst & 1;                      // parity of plane k
      for (int i = 0; i < NI; ++i) {
        asm volatile("" : "+r"(oT));
        const int bn = odd ? 0 : BUF;          // half of the exchange block of plane k-1
        if (i >= I0 && i <= IZ1 + 1) {
          const int cp = odd ? 0 : C::NYP;     // fields of the copy of plane k-1
          const T *a0 = s_a0 + cp * TLE + oT;
          V outm[10];
          cstage(s_ap + cp * YPF + oT, s_am + cp * YPF + oT, [&](int q) { return lds_pair(a0 + q * TLE); }, accA, accB, outm);
          // a4, a6, a9: u_b = m'/rho', u' = u_b + F/rho', Pi^neq' = Pi' - rho' u_b u_b (Hermite form)
          if ((unsigned)(i + ju) < (unsigned)njs) {
            const V rinv = prcp<T>(outm[0] + V(T(1)));
            const V ubx = outm[1] * rinv, uby = outm[2] * rinv, ubz = outm[3] * rinv;
            V o[NF_MAX];
            o[0] = outm[0];
            o[1] = pfma(Fr[0], rinv, ubx);
            o[2] = pfma(Fr[1], rinv, uby);
            o[3] = pfma(Fr[2], rinv, ubz);
            o[4] = outm[4] - outm[1] * ubx;
            o[5] = outm[5] - outm[2] * uby;
            o[6] = outm[6] - outm[3] * ubz;
            o[7] = outm[7] - outm[1] * uby;
            o[8] = outm[8] - outm[1] * ubz;
            o[9] = outm[9] - outm[2] * ubz;
            store_pair<T, FM_FLOW, SLAB>(P, o, pst, kst + i - 2, gx_, gy_, img0, fs);
          }
        }
        if (i <= IZ1 && i >= I0 + 1) phase_D(IC<0>(), oZ, oT, s, bn, eoff, emask, esign, Fr);
        pst += L.plane;
        odd = !odd;
        iter_end(IC<0>(), i);
      }
    } else {
    // ============================ halo-column warp ============================
    // node pairs: lanes 0 .. 2 RY - 1 own the two halo columns; every lane owns a pair of the halo rows
    PhaseState<T> pc, ph_;
    pc.clear(); ph_.clear();
    const int cl = c0 > 0 ? c0 - 1 : 0, cr = c0 + 2 < RX ? c0 + 2 : RX - 1;   // clamped: unused halves
    const int rh = hi ? 0 : RY - 1, ch = HL + 2 * lx;
    const PairGeom gc = {r * RX, c0, cl, cr, 0, r * FQW + (c0 - (HL - 2)) / 2, 0, 0};
    const PairGeom gh = {rh * RX, ch, ch - 1, ch + 2, rh * ZW + 2 + 2 * lx, rh * FQW + 1 + lx, rh * TX + 2 * lx, 0};
    bool odd = kst & 1;                      // parity of plane k
    for (int i = 0; i < NI; ++i) {
      const int bo = odd ? BUF : 0, bn = BUF - bo;
      if (i >= (TWO ? 0 : 1) && i <= IZ1) mbar_wait(&bars[s], mph);
      if (i >= I0 - 2 && i <= IZ1 - 1) {
        // x-pass terms of the two halo columns x0-1 (its a+) and x0+TX (its a-) of every region row of
        // plane k+1 (moments in the next ring slot), one iteration ahead of the rows that use them
        const int s1 = s == S - 1 ? 0 : s + 1;
        mbar_wait(&bars[s1], s1 == 0 ? mph ^ 1u : mph);
        if (lane < 2 * RY) {
          const T *p = mom_at(s1) + r * RX + (cside ? HL + TX : HL - 1);
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
          T *xh = (cside ? s_am : s_ap) + TY * TX + (odd ? 0 : RY) + r;      // parity of plane k+1
#pragma unroll
          for (int g = 0; g < 8; ++g) xh[g * YPF] = cside ? gm[g] : gp[g];
        }
      }
      if (TWO && i <= IZ1) {
        if (lane < 2 * RY) phase_B(IC<2>(), IC<0>(), pc, gc, s, bo, bn);
        if (!UNI) phase_B(IC<1>(), IC<0>(), ph_, gh, s, bo, bn);   // (UNI: a phase warp owns the halo rows)
      }
      odd = !odd;
      iter_end(IC<1>(), i);
    }
    }
  } else {
    // ============================ phase warps ============================
    if (UNI) asm volatile("setmaxnreg.dec.sync.aligned.u32 136;");
    PhaseState<T> p0, p1;     // two node pairs: rows r and r + 2 (UNI: one)
    p0.clear(); p1.clear();
    const int oZ = r * ZW + 2 + 2 * lx, oF = r * FQW + 1 + lx, oG = r * TX + 2 * lx;
    const PairGeom g0 = {r * RX, c0, c0 - 1, c0 + 2, oZ, oF, oG, oT};
    // the halo column's z-combinations of n for the lanes at the tile edge (row r of the raw array of that
    // side), zeros for every other lane; the lane's weights of that share
    const int eoff = (lx == 0 ? C::B_ZL : (lx == LX - 1 ? C::B_ZL + RY : C::B_ZZ)) + 2 + r;
    const V emask(lx == 0 ? T(1) : T(0), lx == LX - 1 ? T(1) : T(0));
    const T esign = lx == 0 ? T(-0.5) : T(0.5);
    // planes whose phi' the thread stores (rows r and r + 2): its chunk, without the imposed inflow / outflow
    // planes; nothing when the node belongs to the neighbouring (shifted-back) tile
    const int pjlo = max(z0, P.jet_lo ? 1 : 0);
    const int pnj = min(z1, P.out_hi ? L.nz - 1 : L.nz) - pjlo;
    const int pnjs0 = (!phalo && gx_ >= xs && gy_ >= ys) ? pnj : 0, pnjs1 = (gx_ >= xs && gy_ + 2 >= ys) ? pnj : 0;
    T *pph = P.out.f[F_PHI] + o00 + (long long)(kst - 1) * L.plane;   // phi of the first pair, plane k-1
    const int pju = kst - 1 - pjlo;          // (plane k-1) - pjlo = i + pju
    int bo = (kst & 1) * BUF;
    for (int i = 0; i < NI; ++i) {
      const int bn = BUF - bo;
      if (i <= IZ1) {
        mbar_wait(&bars[s], mph);
        if (UNI) {
          // one pair per thread; the warp of the halo rows runs the same code and stores nothing
          // (D: the C warps)
          const V f0 = phase_B(IC<0>(), IC<0>(), p0, g0, s, bo, bn);
          const bool in0 = (unsigned)(i + pju) < (unsigned)pnjs0;
          stg_pair_if(in0, pph, f0);
          V o[NF_MAX];
          o[F_PHI] = f0;
          store_images<T, FM_PHI>(o, pph, 0u, img0, in0);       // (pph is the phi array itself: field spacing 0)
          if (SLAB && in0) store_rare<T, FM_PHI, SLAB>(P, o, kst + i - 1, gx_, gy_, false);
        } else {
        if (i >= I0 + 1) phase_D(IC<0>(), g0.oZ, g0.oT, s, bn, eoff, emask, esign, nullptr);   // (rows r + 2: the halo-row warp)
        const V f0 = phase_B(IC<0>(), IC<0>(), p0, g0, s, bo, bn);
        const V f1 = phase_B(IC<0>(), IC<2>(), p1, g0, s, bo, bn);
        // a9: phi'(k-1) of the two pairs
        const bool in0 = (unsigned)(i + pju) < (unsigned)pnjs0, in1 = (unsigned)(i + pju) < (unsigned)pnjs1;
        stg_pair_if(in0, pph, f0);
        stg_pair_if(in1, pph + 2 * L.px, f1);
        V o[NF_MAX];
        o[F_PHI] = f0;
        store_images<T, FM_PHI>(o, pph, 0u, img0, in0);         // (pph is the phi array itself: field spacing 0)
        if (SLAB && in0) store_rare<T, FM_PHI, SLAB>(P, o, kst + i - 1, gx_, gy_, false);
        o[F_PHI] = f1;
        store_images<T, FM_PHI>(o, pph + 2 * L.px, 0u, img1, in1);
        if (SLAB && in1) store_rare<T, FM_PHI, SLAB>(P, o, kst + i - 1, gx_, gy_ + 2, false);
        }
      }
      pph += L.plane;
      bo = bn;
      iter_end(IC<0>(), i);
    }
  }
}

// ------------------------------------------------------------------ host side
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

constexpr int TSLB_MAX_DEVICES = 64;

struct TiledPlan {
  std::string name;
  int precision = 0, tx = 0, ty = 0, zc = 0;
  int device = 0;        // the context's device (kernel attributes are set once per device)
  TiledMaps maps[2];     // per source buffer
  bool two = false;
};

// tile shapes: 32x8 (fp32: ~103 KB of shared memory -> two CTAs per SM, whose barrier phases interleave;
// measured 30.2 vs 27.6 GLUPS for 64x8 on C5); 32x6 for the two-component fp64 build (TileCfg::UNI: three
// flow warps + the halo-row warp are one warpgroup, three phase warps + the halo rows' phase warp another)
constexpr int TILE_TX = 32, TILE_TY = 8, TILE_TY_UNI = 6;
inline void tiled_tile(int precision, bool two, int &tx, int &ty) {
  tx = TILE_TX;
  ty = precision == TSLB_F64 && two ? TILE_TY_UNI : TILE_TY;
}

inline bool tiled_supported(int precision, bool two, int nx, int ny, int nz) {
  int tx, ty;
  tiled_tile(precision, two, tx, ty);
  // rows of the padded arrays must be multiples of 16 bytes for TMA (px = nx + 16)
  return nx % (precision == TSLB_F32 ? 4 : 2) == 0 && nz >= 1 && nx >= tx && ny >= ty &&
         (long long)ny * (nx + 2 * GX) < (1ll << 31);      // (offset of a node's periodic y image: 32 bits)
}

inline bool tiled_plan_create(TiledPlan &pl, int precision, const Layout &L, void *fields[2][NF_MAX], int nfields,
                              int device, std::string &why) {
  pl.device = device;
  PFN_encodeTiled enc = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void **)&enc, cudaEnableDefault, &qres);
  if (e != cudaSuccess || !enc || qres != cudaDriverEntryPointSuccess) {
    why = "cuTensorMapEncodeTiled not available from the driver";
    return false;
  }
  pl.precision = precision;
  pl.two = nfields == 11;
  tiled_tile(precision, pl.two, pl.tx, pl.ty);
  const size_t es = precision == TSLB_F32 ? 4 : 8;
  const CUtensorMapDataType dt = precision == TSLB_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  const int RX = pl.tx + 2 * (es == 4 ? 4 : 2), RY = pl.ty + 2, RYP = pl.ty + 4;
  for (int b = 0; b < 2; ++b) {
    const size_t fstride = (size_t)((char *)fields[b][1] - (char *)fields[b][0]);
    if (fstride % 2 || fstride / 2 > 0xffffffffull) { why = "field arrays more than 8 GB apart"; return false; }
    pl.maps[b].fsh = (unsigned)(fstride / 2);
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
  // z chunking: every chunk pays a 6-iteration pipeline prologue (three of them light), and the grid runs in
  // waves of (CTAs per SM) x (SM count): pick the chunk length that minimises waves x (zc + 5) -- up to 128
  // planes.  Longer chunks save prologue iterations, but CTAs start in blockIdx order whenever a slot frees, so the
  // y-neighbour of a tile (ntx launches later) runs behind it by a fixed fraction of a chunk, and with long chunks
  // its halo rows have left L2 when it reads them (DRAM reads of a C5 step: 22.2 GB at 64 planes, 25.3 at 128, 27.8
  // at 256; profiles/r02_zchunk_sweep.md).  With the final kernels 128 planes measure best on C5 (39.9 against
  // 39.4 GLUPS at 64 and 39.9 at 256, 60 steps).
  const long long tiles = (long long)pl.maps[0].ntx * pl.maps[0].nty;
  int nsm = 148;
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, device);
  const long long slots = (long long)nsm * (precision == TSLB_F32 ? 2 : 1);
  int zc = L.nz;
  long long best = -1;
  for (int cand = 8; cand <= 128; cand *= 2) {
    const int c = cand < L.nz ? cand : L.nz;
    const long long ctas = tiles * ((L.nz + c - 1) / c);
    const long long cost = ((ctas + slots - 1) / slots) * (c + 5);
    if (best < 0 || cost < best) { best = cost; zc = c; }
  }
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
  boundary_node<T>(P, P.in, x, y, z, step_index(P), o, two != 0);
  const long long i0 = ((long long)z * L.py + Y) * L.px + X;
  const int nf = two ? 11 : 10;
  for (int k = 0; k < nf; ++k) P.out.f[k][i0] = o[k];
}

template <typename T, int TX, int TY, bool TWOC>
cudaError_t launch_tiled_t(TiledPlan &pl, const StepParams<T> &P, int src, int order, cudaStream_t st) {
  constexpr bool two = TWOC;
  const bool slab = P.halo_lo || P.halo_hi;
  const TiledMaps &M = pl.maps[src];
  dim3 grid(M.ntx * M.nty, (P.L.nz + M.zc - 1) / M.zc);
  cudaError_t e = cudaSuccess;
#define TSLB_LAUNCH(ORD, SL)                                                                            \
  do {                                                                                                \
    using Cf = TileCfg<T, TX, TY, TWOC>;                                                              \
    auto kern = tiled_step_kernel<T, TX, TY, ORD, TWOC, SL>;                                          \
    static bool attr_set[TSLB_MAX_DEVICES] = {};   /* the attribute is per DEVICE */                  \
    if (pl.device < 0 || pl.device >= TSLB_MAX_DEVICES || !attr_set[pl.device]) {                     \
      e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cf::SMEM_BYTES); \
      if (e != cudaSuccess) return e;                                                                 \
      if (pl.device >= 0 && pl.device < TSLB_MAX_DEVICES) attr_set[pl.device] = true;                 \
    }                                                                                                 \
    kern<<<grid, Cf::NTHREADS, Cf::SMEM_BYTES, st>>>(P, M);                                           \
  } while (0)
  if (slab) { if (order >= 3) TSLB_LAUNCH(3, true); else TSLB_LAUNCH(2, true); }
  else      { if (order >= 3) TSLB_LAUNCH(3, false); else TSLB_LAUNCH(2, false); }
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
  return two ? launch_tiled_t<float, TILE_TX, TILE_TY, true>(pl, P, src, order, st)
             : launch_tiled_t<float, TILE_TX, TILE_TY, false>(pl, P, src, order, st);
}
template <>
inline cudaError_t launch_tiled<double>(TiledPlan &pl, const StepParams<double> &P, int src, int order, bool two, cudaStream_t st) {
  return two ? launch_tiled_t<double, TILE_TX, TILE_TY_UNI, true>(pl, P, src, order, st)
             : launch_tiled_t<double, TILE_TX, TILE_TY, false>(pl, P, src, order, st);
}

}  // namespace tslb
