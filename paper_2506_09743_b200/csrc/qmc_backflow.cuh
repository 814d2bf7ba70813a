// qmc_backflow.cuh -- local energy of a backflow-transformed Slater-Jastrow wavefunction:
//   rt_i = r_i + sum_{j != i} K_BF(r_ij) (r_i - r_j),  K_BF(r) = w / r
// orbitals at rt, Jastrow factor at r.  Every row of a Slater matrix now depends on every electron, so the last two
// terms of F.5 and the cross term of F.4 no longer vanish.  Two kernels, one walker per warp: the
// explicit route (every determinant eliminated on its own) and, below it, the route on the reference's tables.
//
// Formulation (derived here; the oracle evaluates F.3-F.5 coordinate by coordinate instead).  With the 3x3 blocks of
// the map's Jacobian  J_im = d rt_i / d r_m  (pair matrices P_ij = (w/r_ij)(1 - u u^T), u = (r_i - r_j)/r_ij:
// J_ii = 1 + sum_j P_ij, J_im = -P_im), V^a[i][k] = d_a phi_k(rt_i), W^a = V^a A^-1 (electrons x electrons, per
// determinant and spin) and  C_ii' = sum_m J_im J_i'm  (3x3 blocks, electrons of both spins):
//   sum_l Tr(A^-1 d_l A) gJ_l             = sum_i  W_ii . gt_i,        gt_i = sum_m J_im grad_m J
//   sum_l Tr(A^-1 d_l^2 A)                = Tr(A^-1 Bt),   Bt[i][k] = C_ii : Hess phi_k(rt_i) + L_i . grad phi_k(rt_i),
//                                           L_i = sum_l d^2 rt_i / d x_l^2 = -4 w sum_j (r_i - r_j)/r_ij^3
//   sum_l [Tr(A^-1 d_l A)^2 - Tr((A^-1 d_l A)^2)]  and the up-down cross term of F.4, together
//       E2 = sum_{i,i'} sum_{a,a'} C_ii'[a][a'] ( W^a_ii W^a'_i'i' - [same spin] W^a_ii' W^a'_i'i )
// so that, with the per-row operator B = -1/2 Bt - gt_i . grad phi (folded at AO level as in the plain path),
//   -1/2 lap Psi / Psi = -1/2 (lap J + |grad J|^2) + sum_n w_n [ Tr(A_n^-1 B_n)^up + Tr(..)^dn - 1/2 E2_n ] / sum_n w_n.
// Without backflow C is the identity and E2 = 0 (G.5/G.6).
#pragma once
#include <type_traits>

#include "qmc_device.cuh"
#include "qmc_eval.cuh"  // een_terms_inl / een_param_terms_inl (D.3)

namespace qmc {

// symmetric 3x3 in the order {xx, yy, zz, xy, yz, zx}
struct Sym3 { double xx, yy, zz, xy, yz, zx; };
__device__ __forceinline__ void sym_mul(const Sym3 &a, const Sym3 &b, double o[9]) {  // o = a b, row-major (not symmetric)
  const double A[3][3] = {{a.xx, a.xy, a.zx}, {a.xy, a.yy, a.yz}, {a.zx, a.yz, a.zz}};
  const double B[3][3] = {{b.xx, b.xy, b.zx}, {b.xy, b.yy, b.yz}, {b.zx, b.yz, b.zz}};
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) o[3 * i + j] = fma(A[i][0], B[0][j], fma(A[i][1], B[1][j], A[i][2] * B[2][j]));
}

constexpr int kBfLP = 8;  // lanes per (determinant, spin) problem: n_up, n_dn <= 8
// fallback thresholds of the table route (as kFallbackK / kFallbackKappa of the plain path, tighter: the second-order
// tables carry one more factor A0^-1), not scaled with |E_L|.  Measured (table route against the explicit route, 32768
// equilibrated CO walkers / worst of 100 random systems against the long-double CPU reference): 1e4 scaled with
// max(1, |E_L|): 2.3e-8 / 1.8e-8, 2.8 ms; 1e4: 1.4e-9 / 6.4e-10, 3.4 ms; 1e3: 6e-11 / 2e-10, 4.9 ms.
#ifndef QMC_BF_FALLBACK_K
#define QMC_BF_FALLBACK_K 1.0e4
#endif
#ifndef QMC_BF_FALLBACK_KAPPA
#define QMC_BF_FALLBACK_KAPPA 1.0e4
#endif
#ifndef QMC_BF_FALLBACK_ESCALE
#define QMC_BF_FALLBACK_ESCALE 0  // 1: thresholds times max(1, |E_L|) as in the plain path -- measured too lenient here
#endif
constexpr double kBfFallbackK = QMC_BF_FALLBACK_K, kBfFallbackKappa = QMC_BF_FALLBACK_KAPPA;

template <int NS, int NMO>
struct BfGeo {
  static constexpr int NE = 2 * NS;
  static constexpr int oXYZ = 0;                       // [3][32] electron coordinates
  static constexpr int oGJ = oXYZ + 96;                // [3][32] grad_i J
  static constexpr int oS = oGJ + 96;                  // [6][32] S_i = sum_j P_ij
  static constexpr int oC = oS + 192;                  // [NE (NE + 1) / 2][9] C blocks C_ii', i <= i' (C_i'i is the transpose)
  static constexpr int oMO = oC + NE * (NE + 1) / 2 * 9;  // [5][NE][NMO] MO rows: value, operator, d_x, d_y, d_z
  static constexpr int oW = oMO + 5 * NE * NMO;        // [4][3][NS][NS] W^a of the four problems in flight
  static constexpr int oPr = oW + 4 * 3 * NS * NS;     // [4][2] {det, trace}
  static constexpr int oP = oPr + 8;                   // [NE (NE - 1) / 2][6] pair matrices (P_im = P_mi)
  static constexpr int total = (oP + cmax(NE * (NE - 1) / 2, 1) * 6 + 1) & ~1;
  static constexpr bool kTab = false;
  __device__ static __forceinline__ int pofs(int i, int m, int ne) {
    const int a = min(i, m), b = max(i, m);
    return ((a * (2 * ne - a - 1)) / 2 + (b - a - 1)) * 6;
  }
  __device__ static __forceinline__ int cofs(int a, int b, int ne) {  // a <= b
    return (a * ne - (a * (a - 1)) / 2 + (b - a)) * 9;
  }
};

// Scratch of the table route (backflow_tables_kernel): no off-diagonal C blocks (the same-spin ones are formed pair by
// pair where they are contracted, the cross-spin ones enter only through t0), each pair matrix once (P_im = P_mi).
// Per spin, with row stride 8:  T [NS][8], M1 [NS][8] (first-order table of the combined operator), rho = A0^-1 [NS][8],
// G = A0^-1 B0 [NS][8], W0 [3][NS][8], m [3][NS][8], Y2 [kMaxVirt(q)][8(p)]; then scalars [8].
template <int NS, int NMO>
struct BfGeoT {
  static constexpr int NE = 2 * NS;
  static constexpr int oXYZ = 0;                       // [3][32] electron coordinates
  static constexpr int oGJ = oXYZ + 96;                // [3][32] grad_i J
  static constexpr int oS = oGJ + 96;                  // [6][32] S_i = sum_j P_ij
  static constexpr int oCd = oS + 192;                 // [6][32] diagonal blocks C_ii (symmetric)
  static constexpr int oMO = oCd + 192;                // [5][NE][NMO] MO rows, later R [2][3][NS][8]
  static constexpr int oP = oMO + cmax(5 * NE * NMO, 2 * 3 * NS * 8);  // [NE (NE - 1) / 2][6] pair matrices
  static constexpr int tSpin = 4 * NS * 8 + 2 * 3 * NS * 8 + kMaxVirt * 8;
  static constexpr int oTab = oP + cmax(NE * (NE - 1) / 2, 1) * 6;
  static constexpr int oSc = oTab + 2 * tSpin;
  static constexpr int total = (oSc + 16 + 1) & ~1;  // scalars [16]: per spin {det, t0, s0, kappa}, then t_w per spin
  static constexpr int NC = 3 * NE;                    // coordinates l = 3 m + b
  static constexpr int LS = (NC + 3) & ~3;             // stride of an E vector in the global scratch
  static constexpr int eDoubles = 2 * kMaxVirt * NS * LS;  // E[sp][q][p][l] per warp (global memory, L2-resident)
  static constexpr bool kTab = true;
  __device__ static __forceinline__ int pofs(int i, int m, int ne) {
    const int a = min(i, m), b = max(i, m);
    return ((a * (2 * ne - a - 1)) / 2 + (b - a - 1)) * 6;
  }
};

// C_ii' = sum_m J_im J_i'm for i != i' (3x3, row-major into cc):  -J_ii P_ii' - P_ii' J_i'i' + sum_{m != i, i'} P_im P_i'm
// from the pair matrices and their sums in the warp's scratch (J_ii = 1 + S_i, J_im = -P_im).
template <class BG>
__device__ __forceinline__ void bf_pair_block(const double *__restrict__ sP, const double *__restrict__ sS, int gi, int gi2, int ne,
                                              double cc[9]) {
  const double *pq = sP + BG::pofs(gi, gi2, ne);
  const Sym3 Pq{pq[0], pq[1], pq[2], pq[3], pq[4], pq[5]};
  const Sym3 J1{1.0 + sS[gi], 1.0 + sS[32 + gi], 1.0 + sS[64 + gi], sS[96 + gi], sS[128 + gi], sS[160 + gi]};
  const Sym3 J2{1.0 + sS[gi2], 1.0 + sS[32 + gi2], 1.0 + sS[64 + gi2], sS[96 + gi2], sS[128 + gi2], sS[160 + gi2]};
  double t[9];
  sym_mul(J1, Pq, cc);
  sym_mul(Pq, J2, t);
#pragma unroll
  for (int k = 0; k < 9; ++k) cc[k] = -cc[k] - t[k];
  for (int m = 0; m < ne; ++m) {
    if (m == gi || m == gi2) continue;
    const double *p1 = sP + BG::pofs(gi, m, ne), *p2 = sP + BG::pofs(gi2, m, ne);
    sym_mul(Sym3{p1[0], p1[1], p1[2], p1[3], p1[4], p1[5]}, Sym3{p2[0], p2[1], p2[2], p2[3], p2[4], p2[5]}, t);
#pragma unroll
    for (int k = 0; k < 9; ++k) cc[k] += t[k];
  }
}

// Phases 1-2 of a backflow evaluation for walker w (one warp; lane = electron): Jastrow, potential, the backflow map and its
// derivatives (pair matrices P, their sums S, the C blocks) and the five MO planes at the backflow coordinates (value,
// combined operator B = -1/2 (C_ii : Hess + L_i . grad) - gt_i . grad, d_x, d_y, d_z) into the warp's scratch.
// Jsh / esh: this lane's share of J and of -1/2 (lap J + |grad J|^2) + V_ee + V_en.
// MB: the wavefunction carries the many-body Jastrow kernels D.2 / D.3 (own instantiations: their code costs the plain
// ones 6 % when it is merely present).  DERIV: also the parameter derivatives of J into io.O and d rt / d w into the grad J region.
template <int NS, int NMO, class BG, bool DERIV = false, bool MB = false>
__device__ __forceinline__ void bf_build(const SysParams &P, const double *__restrict__ sCf, const double *__restrict__ sExp,
                                         double *__restrict__ ws, const WalkerIO &io, int64_t w, int lane, double &Jsh, double &esh) {
  constexpr int NT = (NMO + 7) / 8;
  double *sXYZ = ws + BG::oXYZ, *sGJ = ws + BG::oGJ, *sS = ws + BG::oS, *sMO = ws + BG::oMO, *sP = ws + BG::oP;
  const int n_up = P.n_up, ne = P.n_e;
  const double bw = P.bf_w;
  const bool act = lane < ne;
  const int i = act ? lane : 0;
  {
    double x = 0.37 + 0.11 * lane, y = -0.21 + 0.07 * lane, z = 0.53 - 0.05 * lane;
    if (act) {
      x = io.r_in[((int64_t)lane * 3 + 0) * io.M + w];
      y = io.r_in[((int64_t)lane * 3 + 1) * io.M + w];
      z = io.r_in[((int64_t)lane * 3 + 2) * io.M + w];
    }
    sXYZ[lane] = x; sXYZ[32 + lane] = y; sXYZ[64 + lane] = z;
    __syncwarp();
    // ---- phase 1: Jastrow (D.1), e-e and e-n potential (eq. 1), the backflow map and its derivatives
    double Jp = 0.0, gJx = 0.0, gJy = 0.0, gJz = 0.0, lapJ = 0.0, vee = 0.0, ven = 0.0;
    if (MB && P.n_een > 0) {
      // electron-electron-nucleus kernel (D.3): this electron's share, and with DERIV the seven parameters
      // of every term summed over the walker's electrons.  First, while little is live.
      double t[5];
      een_terms_inl<true>(P, sXYZ, 0, ne, i, x, y, z, t);
      Jp = t[0]; gJx = t[1]; gJy = t[2]; gJz = t[3]; lapJ = t[4];
      if (DERIV) {
        double *row = io.O ? io.O + w * (int64_t)(kJastrowParams + 7 * P.n_een + P.n_det_all + 1) : nullptr;
        for (int mu = 0; mu < P.n_een; ++mu) {
          double dq[7];
          een_param_terms_inl(P, sXYZ, 0, ne, i, x, y, z, mu, dq);
#pragma unroll
          for (int k = 0; k < 7; ++k) {
            double tk = act ? dq[k] : 0.0;
#pragma unroll
            for (int mm = 16; mm > 0; mm >>= 1) tk += shfl_xor_d(tk, mm);
            if (lane == 0 && row) row[kJastrowParams + 7 * mu + k] = tk;
          }
        }
      }
    }
    double px = 0.0, py = 0.0, pz = 0.0, Lx = 0.0, Ly = 0.0, Lz = 0.0;
    Sym3 S{0, 0, 0, 0, 0, 0}, S2{0, 0, 0, 0, 0, 0};
    double dpar = 0.0, danti = 0.0, dbb = 0.0, dw0 = 0.0, dw1 = 0.0, dw2 = 0.0;  // DERIV: parameter derivatives of J
    const bool up = i < n_up;
    for (int o = 1; o < ne; ++o) {
      int j = i + o;
      j -= (j >= ne) ? ne : 0;
      const double dx = x - sXYZ[j], dy = y - sXYZ[32 + j], dz = z - sXYZ[64 + j];
      const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
      const double ri = rsqrt_fast(r2), r = r2 * ri;
      const double a = ((j < n_up) == up) ? P.a_par : P.a_anti;
      const double di = rcp_fast(fma(P.b, r, 1.0));
      const double u1 = a * di * di, u2 = -2.0 * P.b * u1 * di;
      Jp = fma(0.5 * a * di, r, Jp);
      if (DERIV) {  // D.1: dK/da = r / (1 + b r), dK/db = -a r^2 / (1 + b r)^2; every pair is met by both of its lanes
        const double rd = 0.5 * r * di;
        if ((j < n_up) == up) dpar += rd; else danti += rd;
        dbb = fma(-a * rd, r * di, dbb);
      }
      const double sc = u1 * ri;
      gJx = fma(sc, dx, gJx); gJy = fma(sc, dy, gJy); gJz = fma(sc, dz, gJz);
      lapJ += fma(2.0, sc, u2);
      vee = fma(0.5, ri, vee);
      const double ux = dx * ri, uy = dy * ri, uz = dz * ri, eta = bw * ri;
      px += ux; py += uy; pz += uz;
      Sym3 Pm{eta * (1.0 - ux * ux), eta * (1.0 - uy * uy), eta * (1.0 - uz * uz), -eta * ux * uy, -eta * uy * uz, -eta * uz * ux};
      S.xx += Pm.xx; S.yy += Pm.yy; S.zz += Pm.zz; S.xy += Pm.xy; S.yz += Pm.yz; S.zx += Pm.zx;
      S2.xx = fma(eta, Pm.xx, S2.xx); S2.yy = fma(eta, Pm.yy, S2.yy); S2.zz = fma(eta, Pm.zz, S2.zz);
      S2.xy = fma(eta, Pm.xy, S2.xy); S2.yz = fma(eta, Pm.yz, S2.yz); S2.zx = fma(eta, Pm.zx, S2.zx);
      const double l3 = -4.0 * bw * ri * ri * ri;
      Lx = fma(l3, dx, Lx); Ly = fma(l3, dy, Ly); Lz = fma(l3, dz, Lz);
      if (act && j > i) {  // each pair matrix once (P_ij = P_ji)
        double *pp = sP + BG::pofs(i, j, ne);
        pp[0] = Pm.xx; pp[1] = Pm.yy; pp[2] = Pm.zz; pp[3] = Pm.xy; pp[4] = Pm.yz; pp[5] = Pm.zx;
      }
    }
    for (int at = 0; at < P.n_atoms; ++at) {
      const double dx = x - P.atom[at][0], dy = y - P.atom[at][1], dz = z - P.atom[at][2];
      const double d2 = fma(dx, dx, fma(dy, dy, dz * dz)), rinv = rsqrt_fast(d2);
      ven = fma(-P.atom[at][3], rinv, ven);
      if ((MB && P.has_en) || DERIV) {
        // electron-nucleus Jastrow kernel (D.2): K = N / D, N = w0 r + w1 r^2, D = 1 + w2 r,
        // K' = (N' - w2 K) / D, K'' = (N'' - 2 w2 K') / D; grad_i J += K' d / r, lap_i J += K'' + 2 K' / r
        const double ra = d2 * rinv, Di = rcp_fast(fma(P.en_w2, ra, 1.0));
        const double K = ra * fma(P.en_w1, ra, P.en_w0) * Di;
        if (MB && P.has_en) {
          const double K1 = (fma(2.0 * P.en_w1, ra, P.en_w0) - P.en_w2 * K) * Di;
          const double K2 = 2.0 * fma(-P.en_w2, K1, P.en_w1) * Di;
          const double sc = K1 * rinv;
          Jp += K;
          gJx = fma(sc, dx, gJx); gJy = fma(sc, dy, gJy); gJz = fma(sc, dz, gJz);
          lapJ += fma(2.0, sc, K2);
        }
        if (DERIV) {  // dK/dw0 = r / D, dK/dw1 = r^2 / D, dK/dw2 = -N r / D^2 = -K r / D
          const double rd = ra * Di;
          dw0 += rd;
          dw1 = fma(ra, rd, dw1);
          dw2 = fma(-K, rd, dw2);
        }
      }
    }

    if (DERIV) {
      if (!act) dpar = danti = dbb = dw0 = dw1 = dw2 = 0.0;
#pragma unroll
      for (int mm = 16; mm > 0; mm >>= 1) {
        dpar += shfl_xor_d(dpar, mm); danti += shfl_xor_d(danti, mm); dbb += shfl_xor_d(dbb, mm);
        dw0 += shfl_xor_d(dw0, mm); dw1 += shfl_xor_d(dw1, mm); dw2 += shfl_xor_d(dw2, mm);
      }
      double *row = io.O ? io.O + w * (int64_t)(kJastrowParams + 7 * P.n_een + P.n_det_all + 1) : nullptr;
      if (lane == 0 && row) {
        row[0] = dpar; row[1] = danti; row[2] = dbb; row[3] = dw0; row[4] = dw1; row[5] = dw2;
      }
    }
    const double xt = fma(bw, px, x), yt = fma(bw, py, y), zt = fma(bw, pz, z);
    sGJ[lane] = gJx; sGJ[32 + lane] = gJy; sGJ[64 + lane] = gJz;
    sS[lane] = S.xx; sS[32 + lane] = S.yy; sS[64 + lane] = S.zz; sS[96 + lane] = S.xy; sS[128 + lane] = S.yz; sS[160 + lane] = S.zx;
    __syncwarp();
    // gt_i = sum_m J_im grad_m J = (1 + S_i) grad_i J - sum_{m != i} P_im grad_m J
    double gtx = gJx + fma(S.xx, gJx, fma(S.xy, gJy, S.zx * gJz));
    double gty = gJy + fma(S.xy, gJx, fma(S.yy, gJy, S.yz * gJz));
    double gtz = gJz + fma(S.zx, gJx, fma(S.yz, gJy, S.zz * gJz));
    const Sym3 Ji{1.0 + S.xx, 1.0 + S.yy, 1.0 + S.zz, S.xy, S.yz, S.zx};
    for (int m = 0; m < ne; ++m) {
      if (m == i) continue;
      const double *pp = sP + BG::pofs(i, m, ne);
      const double ax = sGJ[m], ay = sGJ[32 + m], az = sGJ[64 + m];
      gtx -= fma(pp[0], ax, fma(pp[3], ay, pp[5] * az));
      gty -= fma(pp[3], ax, fma(pp[1], ay, pp[4] * az));
      gtz -= fma(pp[5], ax, fma(pp[4], ay, pp[2] * az));
    }
    // C blocks of row i:  C_ii = (1 + S_i)^2 + sum_m P_im^2 (P^2 = (w/r) P),
    //   C_ii' = -(1 + S_i) P_ii' - P_ii' (1 + S_i') + sum_{m != i, i'} P_im P_i'm
    Sym3 Cd;
    {
      double q[9];
      sym_mul(Ji, Ji, q);
      Cd = Sym3{q[0] + S2.xx, q[4] + S2.yy, q[8] + S2.zz, q[1] + S2.xy, q[5] + S2.yz, q[2] + S2.zx};
    }
    if constexpr (BG::kTab) {  // the diagonal blocks only (backflow_tables_kernel forms the others where it contracts them)
      double *sCd = ws + BG::oCd;
      sCd[lane] = Cd.xx; sCd[32 + lane] = Cd.yy; sCd[64 + lane] = Cd.zz; sCd[96 + lane] = Cd.xy; sCd[128 + lane] = Cd.yz; sCd[160 + lane] = Cd.zx;
    } else {
      // every block C_ii', i <= i' (the explicit kernel's E2 runs over all pairs of both spins): the diagonal by its lane, the
      // others one lane per unordered pair
      double *sCb = ws + BG::oC;
      if (act) {
        double *cb = sCb + BG::cofs(i, i, ne);
        cb[0] = Cd.xx; cb[1] = Cd.xy; cb[2] = Cd.zx; cb[3] = Cd.xy; cb[4] = Cd.yy; cb[5] = Cd.yz; cb[6] = Cd.zx; cb[7] = Cd.yz; cb[8] = Cd.zz;
      }
      for (int pi = lane; pi < ne * (ne - 1) / 2; pi += 32) {
        int rem = pi, a = 0;
        while (rem >= ne - 1 - a) { rem -= ne - 1 - a; ++a; }
        const int b = a + 1 + rem;  // a < b < ne
        double cc[9];
        bf_pair_block<BG>(sP, sS, a, b, ne, cc);
        double *co = sCb + BG::cofs(a, b, ne);
#pragma unroll
        for (int k = 0; k < 9; ++k) co[k] = cc[k];
      }
    }
    __syncwarp();
    if (DERIV) {  // d rt_i / d w = sum_j (r_i - r_j) / r_ij takes the place of grad J (dead from here on)
      sGJ[lane] = px; sGJ[32 + lane] = py; sGJ[64 + lane] = pz;
    }
    // ---- phase 2: STOs at the backflow coordinates and AO -> MO, per electron:
    // value, combined operator b = -1/2 (C_ii : Hess + L_i . grad) - gt_i . grad, and the three gradient components
    {
      double mv[NMO], mb[NMO], mx[NMO], my[NMO], mz[NMO];
#pragma unroll
      for (int k = 0; k < NMO; ++k) mv[k] = mb[k] = mx[k] = my[k] = mz[k] = 0.0;
      const double trC = Cd.xx + Cd.yy + Cd.zz;
      int chunk = 0;
      double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1.0, r = 1.0, ri = 1.0, ux = 0.0, uy = 0.0, uz = 0.0;
      double cux = 0.0, cuy = 0.0, cuz = 0.0, uCu = 0.0;
      for (int s = 0; s < P.n_shell; ++s) {
        const ShellRec &sh = P.shells[s];
        const int meta = sh.meta, kind = meta & 15;
        if (kind == SH_POW) continue;  // the radial power is in the shell records' own meta word
        if (kind == SH_ATOM) {
          dx = xt - sh.zeta; dy = yt - sh.c1; dz = zt - sh.c2;
          r2 = fma(dx, dx, fma(dy, dy, dz * dz));
          ri = rsqrt_fast(r2);
          r = r2 * ri;
          ux = dx * ri; uy = dy * ri; uz = dz * ri;
          cux = fma(Cd.xx, ux, fma(Cd.xy, uy, Cd.zx * uz));
          cuy = fma(Cd.xy, ux, fma(Cd.yy, uy, Cd.yz * uz));
          cuz = fma(Cd.zx, ux, fma(Cd.yz, uy, Cd.zz * uz));
          uCu = fma(ux, cux, fma(uy, cuy, uz * cuz));
          continue;
        }
        double f = exp_neg(-sh.zeta * r, sExp, P.mc);
        if (meta & kMetaK1) f *= r;
        if (meta & kMetaK2) f *= r2;
        const double rho = fma(sh.kd, ri, -sh.zeta);
        const double F2 = fma(rho, rho, -sh.kd * ri * ri);
        const int row = (meta >> 12) & 15, m = (meta >> 8) & 15;
        int nf = 1, first = 0;
        if (kind == SH_P) nf = 3;
        if (kind == SH_D) nf = 5;
        if (kind == SH_P1 || kind == SH_D1) first = m;
        const int l = (kind == SH_S) ? 0 : ((kind == SH_P || kind == SH_P1) ? 1 : 2);
        for (int t = 0; t < nf; ++t) {
          const int mm = first + t;
          // S, grad S, C : Hess S for the harmonic (l, mm)
          double Sv = 1.0, Sx = 0.0, Sy = 0.0, Sz = 0.0, CS2 = 0.0;
          if (l == 1) {
            Sv = (mm == 0) ? dx : ((mm == 1) ? dy : dz);
            Sx = (mm == 0); Sy = (mm == 1); Sz = (mm == 2);
          } else if (l == 2) {
            if (mm == 0) { Sv = dx * dy; Sx = dy; Sy = dx; CS2 = 2.0 * Cd.xy; }
            else if (mm == 1) { Sv = dy * dz; Sy = dz; Sz = dy; CS2 = 2.0 * Cd.yz; }
            else if (mm == 2) { Sv = dz * dx; Sx = dz; Sz = dx; CS2 = 2.0 * Cd.zx; }
            else if (mm == 3) { Sv = fma(dx, dx, -dy * dy); Sx = 2.0 * dx; Sy = -2.0 * dy; CS2 = 2.0 * (Cd.xx - Cd.yy); }
            else { Sv = fma(2.0 * dz, dz, -fma(dx, dx, dy * dy)); Sx = -2.0 * dx; Sy = -2.0 * dy; Sz = 4.0 * dz; CS2 = 2.0 * (2.0 * Cd.zz - Cd.xx - Cd.yy); }
          }
          const double gx = f * fma(Sv * rho, ux, Sx), gy = f * fma(Sv * rho, uy, Sy), gz = f * fma(Sv * rho, uz, Sz);
          const double sCu = fma(Sx, cux, fma(Sy, cuy, Sz * cuz));  // grad S . C u
          const double CH = f * (CS2 + 2.0 * rho * sCu + Sv * fma(F2, uCu, rho * ri * (trC - uCu)));
          const double val = f * Sv;
          const double bop = fma(-0.5, CH + fma(Lx, gx, fma(Ly, gy, Lz * gz)), -fma(gtx, gx, fma(gty, gy, gtz * gz)));
          const int rw = row + t;
#pragma unroll
          for (int k = 0; k < NMO; ++k) {
            const double cf = sCf[chunk * ((kChunk / 4) * NT * 32) + (((rw >> 2) * NT) + (k >> 3)) * 32 + 4 * (k & 7) + (rw & 3)];
            mv[k] = fma(cf, val, mv[k]);
            mb[k] = fma(cf, bop, mb[k]);
            mx[k] = fma(cf, gx, mx[k]);
            my[k] = fma(cf, gy, my[k]);
            mz[k] = fma(cf, gz, mz[k]);
          }
        }
        if (meta >> 20) ++chunk;
      }
      if (act) {
#pragma unroll
        for (int k = 0; k < NMO; ++k) {
          sMO[(0 * BG::NE + i) * NMO + k] = mv[k];
          sMO[(1 * BG::NE + i) * NMO + k] = mb[k];
          sMO[(2 * BG::NE + i) * NMO + k] = mx[k];
          sMO[(3 * BG::NE + i) * NMO + k] = my[k];
          sMO[(4 * BG::NE + i) * NMO + k] = mz[k];
        }
      }
    }
    __syncwarp();
    Jsh = act ? Jp : 0.0;
    esh = act ? fma(-0.5, lapJ + fma(gJx, gJx, fma(gJy, gJy, gJz * gJz)), vee + ven) : 0.0;
  }
}

template <int NS, int NMO, int WPB, bool DERIV = false, bool MB = false>
__global__ void __launch_bounds__(WPB * 32, 1)
    backflow_energy_kernel(const __grid_constant__ SysParams P, const WalkerIO io) {
  extern __shared__ __align__(16) unsigned char smem[];
  using BG = BfGeo<NS, NMO>;
  // constants: C fragments and the exp table (the layout of load_constants)
  double *sCf = reinterpret_cast<double *>(smem);
  const int nC = P.c_doubles;
  for (int i = threadIdx.x; i < nC; i += blockDim.x) sCf[i] = P.C[i];
  double *sExp = sCf + nC;
  for (int i = threadIdx.x; i < kExpTab + kRngTab; i += blockDim.x) sExp[i] = P.exp_tab[i];
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double *ws = reinterpret_cast<double *>(smem + P.smem_const_bytes) + warp * BG::total;
  double *sCb = ws + BG::oC, *sMO = ws + BG::oMO, *sW = ws + BG::oW, *sPr = ws + BG::oPr;
  const int n_up = P.n_up, n_dn = P.n_dn, ne = P.n_e;
  // list mode (io.fb_list): only the walkers the table-route kernel flagged (nearly singular reference)
  const int64_t n_work = io.fb_list ? (int64_t)*io.fb_count : io.M;
  const int wpb = (int)(blockDim.x >> 5);  // warps launched per block (<= WPB: as many as shared memory holds)
  for (int64_t wk = (int64_t)blockIdx.x * wpb + warp; wk < n_work; wk += (int64_t)gridDim.x * wpb) {
    const int64_t w = io.fb_list ? (int64_t)io.fb_list[wk] : wk;
    double Js, es;
    bf_build<NS, NMO, BG, DERIV, MB>(P, sCf, sExp, ws, io, w, lane, Js, es);
    // ---- phase 3: every determinant on its own, two at a time (four (determinant, spin) problems of 8 lanes)
    const int c = lane & (kBfLP - 1), slot = lane >> 3, gbase = lane - c;
    const int dsel = slot >> 1, sp = slot & 1;
    const int ns = sp ? n_dn : n_up, e0 = sp ? n_up : 0;
    double sig = 0.0, numk = 0.0, numw = 0.0;
    // DERIV (eq. 6 factors): row of this walker; the Jastrow entries are bf_build's, the CI entries D_n / Sigma
    // and the backflow weight's sum_n d_n D_n [Tr(A_n^-1 d_w A_n)^up + ^dn] / Sigma with d_w A[i][k] = grad phi_k . d rt_i / d w
    const int nj = kJastrowParams + 7 * P.n_een;
    double *orow = (DERIV && io.O) ? io.O + w * (int64_t)(nj + P.n_det_all + 1) : nullptr;
    const double *sPw = ws + BG::oGJ;
    for (int n0 = 0; n0 < P.n_det_all; n0 += 2) {
      const int n = n0 + dsel;
      const bool nvalid = n < P.n_det_all;
      const DetCols dc = P.det_cols[nvalid ? n : 0];
      unsigned long long packed = 0ull;
#pragma unroll
      for (int k = 0; k < kMaxSpin; ++k) packed |= (unsigned long long)(unsigned char)dc.col[sp][k] << (8 * k);
      double a0[NS], b0[NS], bi[NS];
      {
        const bool cA = c < ns;
        const int colA = (int)((packed >> (8 * (c & 7))) & 255ull);
#pragma unroll
        for (int q = 0; q < NS; ++q) {
          const bool rq = q < ns;
          const int row = e0 + (rq ? q : 0);
          a0[q] = (rq && cA) ? sMO[(0 * BG::NE + row) * NMO + colA] : ((q == c) ? 1.0 : 0.0);
          b0[q] = (rq && cA) ? sMO[(1 * BG::NE + row) * NMO + colA] : 0.0;
          bi[q] = (rq && cA && q == c) ? 1.0 : 0.0;
        }
      }
      double det = 1.0;
      int perm[NS];
      int myrow = 0;
      bool used = !(c < NS);
#pragma unroll
      for (int k = 0; k < NS; ++k) {
        unsigned key = used ? 0u : (((unsigned)(__double2hiint(a0[k]) & 0x7fffffff) & ~(unsigned)(kBfLP - 1)) | (unsigned)c);
#pragma unroll
        for (int mm = 1; mm < kBfLP; mm <<= 1) key = max(key, __shfl_xor_sync(0xffffffffu, key, mm));
        const int pl = (int)(key & (unsigned)(kBfLP - 1));
        perm[k] = pl;
        if (c == pl) { used = true; myrow = k; }
        double f[NS];
#pragma unroll
        for (int q = 0; q < NS; ++q) f[q] = __shfl_sync(0xffffffffu, a0[q], gbase + pl);
        const double piv = f[k], inv = 1.0 / piv;
        det *= piv;
        double t = a0[k] * inv;
        a0[k] = t;
#pragma unroll
        for (int q = 0; q < NS; ++q) if (q != k) a0[q] = fma(-f[q], t, a0[q]);
        t = b0[k] * inv;
        b0[k] = t;
#pragma unroll
        for (int q = 0; q < NS; ++q) if (q != k) b0[q] = fma(-f[q], t, b0[q]);
        t = bi[k] * inv;
        bi[k] = t;
#pragma unroll
        for (int q = 0; q < NS; ++q) if (q != k) bi[q] = fma(-f[q], t, bi[q]);
      }
      int inversions = 0;
#pragma unroll
      for (int k = 0; k < NS; ++k)
#pragma unroll
        for (int k2 = k + 1; k2 < NS; ++k2) inversions += (perm[k] > perm[k2]) ? 1 : 0;
      if (inversions & 1) det = -det;
      double t0 = 0.0;
#pragma unroll
      for (int q = 0; q < NS; ++q) if (q == myrow && c < NS) t0 = b0[q];
#pragma unroll
      for (int mm = 1; mm < kBfLP; mm <<= 1) t0 += shfl_xor_d(t0, mm);
      if (c == 0) { sPr[slot * 2 + 0] = det; sPr[slot * 2 + 1] = t0; }
      // W^a[q][c] = sum_k V^a[q][column of position perm[k]] A^-1[perm[k]][electron c]   (lane c = electron c of this spin)
      if (c < NS) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          double wq[NS];
#pragma unroll
          for (int q = 0; q < NS; ++q) wq[q] = 0.0;
#pragma unroll
          for (int k = 0; k < NS; ++k) {
            const bool kv = perm[k] < ns;
            const int colk = (int)((packed >> (8 * (perm[k] & 7))) & 255ull);
            const double ak = bi[k];
#pragma unroll
            for (int q = 0; q < NS; ++q)
              if (kv && q < ns) wq[q] = fma(sMO[((2 + a) * BG::NE + e0 + q) * NMO + colk], ak, wq[q]);
          }
#pragma unroll
          for (int q = 0; q < NS; ++q) sW[((slot * 3 + a) * NS + q) * NS + c] = wq[q];
        }
      }
      __syncwarp();
      // E2 of this determinant: lane ld of its 16 lanes = electron ld (both spins)
      const int ld = lane & 15, dme = lane >> 4;  // dme = which of the two determinants
      double e2 = 0.0, tw = 0.0;
      if (ld < ne) {
        const int spi = (ld < n_up) ? 0 : 1, ii = ld - (spi ? n_up : 0);
        const double *Wi = sW + ((dme * 2 + spi) * 3) * NS * NS;
        const double wi[3] = {Wi[(0 * NS + ii) * NS + ii], Wi[(1 * NS + ii) * NS + ii], Wi[(2 * NS + ii) * NS + ii]};
        if (DERIV) tw = fma(sPw[ld], wi[0], fma(sPw[32 + ld], wi[1], sPw[64 + ld] * wi[2]));
        for (int j = 0; j < ne; ++j) {
          const int spj = (j < n_up) ? 0 : 1, jj = j - (spj ? n_up : 0);
          const double *Wj = sW + ((dme * 2 + spj) * 3) * NS * NS;
          const bool lo = ld <= j;  // stored block C_ab, a <= b; C_ba is its transpose
          const double *cb = sCb + BG::cofs(lo ? ld : j, lo ? j : ld, ne);
          const double wj[3] = {Wj[(0 * NS + jj) * NS + jj], Wj[(1 * NS + jj) * NS + jj], Wj[(2 * NS + jj) * NS + jj]};
          double t = 0.0;
#pragma unroll
          for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) t = fma(cb[lo ? 3 * a + b : 3 * b + a] * wi[a], wj[b], t);
          if (spi == spj) {
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
              for (int b = 0; b < 3; ++b) t = fma(-cb[lo ? 3 * a + b : 3 * b + a] * Wi[(a * NS + ii) * NS + jj], Wj[(b * NS + jj) * NS + ii], t);
          }
          e2 += t;
        }
      }
#pragma unroll
      for (int mm = 8; mm > 0; mm >>= 1) e2 += shfl_xor_d(e2, mm);
      if (DERIV) {
#pragma unroll
        for (int mm = 8; mm > 0; mm >>= 1) tw += shfl_xor_d(tw, mm);
      }
      if (ld == 0 && (n0 + dme) < P.n_det_all) {
        const double dd = sPr[(dme * 2) * 2 + 0] * sPr[(dme * 2 + 1) * 2 + 0];
        const double wn = P.det_cols[n0 + dme].d * dd;
        sig += wn;                                                                            // eq. 4
        numk = fma(wn, sPr[(dme * 2) * 2 + 1] + sPr[(dme * 2 + 1) * 2 + 1] - 0.5 * e2, numk);  // F.2, F.4, F.5
        if (DERIV) {
          numw = fma(wn, tw, numw);
          if (orow) orow[nj + n0 + dme] = dd;  // D_n^up D_n^dn, divided by Sigma below
        }
      }
      __syncwarp();
    }
    // ---- assembly (F.1, eq. 1): lanes 0 and 16 hold the sums of the even and odd determinants
    sig += __shfl_xor_sync(0xffffffffu, sig, 16);
    numk += __shfl_xor_sync(0xffffffffu, numk, 16);
#pragma unroll
    for (int mm = 16; mm > 0; mm >>= 1) { Js += shfl_xor_d(Js, mm); es += shfl_xor_d(es, mm); }
    if (lane == 0) {
      if (io.logpsi) io.logpsi[w] = Js + log(fabs(sig));
      if (io.sign) io.sign[w] = (sig > 0.0) ? 1.0 : ((sig < 0.0) ? -1.0 : 0.0);
      if (io.eloc) io.eloc[w] = es + numk / sig + P.vnn;
    }
    if (DERIV) {
      numw += __shfl_xor_sync(0xffffffffu, numw, 16);
      const double isig = 1.0 / __shfl_sync(0xffffffffu, sig, 0);
      __syncwarp();  // the determinant products of lanes 0 and 16 are visible to the whole warp
      if (orow) {
        for (int n = lane; n < P.n_det_all; n += 32) orow[nj + n] *= isig;
        if (lane == 0) orow[nj + P.n_det_all] = numw * isig;
      }
    }
    __syncwarp();
  }
}

// One determinant relative to the reference for the table route: substituted positions p and virtual indices q per spin
// (k <= 2 per spin; expansions with more take the explicit kernel).  24 bytes.
struct BfDet {
  double d;
  uint8_t k[2];
  uint8_t p[2][2];
  uint8_t q[2][2];
  uint16_t orig;  // caller's index of the determinant (the records are sorted by class)
  uint8_t pad[4];
};
static_assert(sizeof(BfDet) == 24, "BfDet is read as three 8-byte words");

// Class boundaries of the sorted records: class 3 k_up + k_dn occupies [start[c], start[c + 1]).
struct BfClasses { int start[10]; };

// One spin's share of a determinant in the table route, substitution order K known at compile time: R = det T_PQ,
// Rd = Tr(adj(T_PQ) M1_PQ), trY = Tr(adj(T_PQ) Y2_PQ), e = Tr(adj(T_PQ) E_PQ,l) and dm = det E_PQ,l for this lane's two
// coordinates.
struct BfSpinTerms { double R, Rd, trY, e0, e1, dm0, dm1, Rw; };
template <int K, int NS, int LS, bool DERIV = false>
__device__ __forceinline__ void bf_spin_terms(const double *__restrict__ T, const double *__restrict__ M1, const double *__restrict__ Y2,
                                              const double *__restrict__ Es, unsigned p0, unsigned p1, unsigned q0, unsigned q1,
                                              bool has0, bool has1, int l0, int l1, BfSpinTerms &o,
                                              const double *__restrict__ Mw = nullptr) {
  o.R = 1.0; o.Rd = 0.0; o.trY = 0.0; o.e0 = o.e1 = o.dm0 = o.dm1 = 0.0; o.Rw = 0.0;
  if constexpr (K == 1) {
    o.R = T[p0 * 8 + q0];
    o.Rd = M1[p0 * 8 + q0];
    if (DERIV) o.Rw = Mw[p0 * 8 + q0];
    o.trY = Y2[q0 * 8 + p0];
    const double *e = Es + (q0 * NS + p0) * LS;
    if (has0) o.e0 = __ldcg(e + l0);
    if (has1) o.e1 = __ldcg(e + l1);
  } else if constexpr (K == 2) {
    const double t11 = T[p0 * 8 + q0], t12 = T[p0 * 8 + q1], t21 = T[p1 * 8 + q0], t22 = T[p1 * 8 + q1];
    o.R = fma(t11, t22, -t12 * t21);
    o.Rd = fma(t22, M1[p0 * 8 + q0], fma(t11, M1[p1 * 8 + q1], -fma(t12, M1[p1 * 8 + q0], t21 * M1[p0 * 8 + q1])));
    if (DERIV) o.Rw = fma(t22, Mw[p0 * 8 + q0], fma(t11, Mw[p1 * 8 + q1], -fma(t12, Mw[p1 * 8 + q0], t21 * Mw[p0 * 8 + q1])));
    o.trY = fma(t22, Y2[q0 * 8 + p0], fma(t11, Y2[q1 * 8 + p1], -fma(t12, Y2[q0 * 8 + p1], t21 * Y2[q1 * 8 + p0])));
    const double *e11 = Es + (q0 * NS + p0) * LS, *e12 = Es + (q1 * NS + p0) * LS, *e21 = Es + (q0 * NS + p1) * LS,
                 *e22 = Es + (q1 * NS + p1) * LS;
    if (has0) {
      const double a = __ldcg(e11 + l0), b2 = __ldcg(e12 + l0), c2 = __ldcg(e21 + l0), dd = __ldcg(e22 + l0);
      o.e0 = fma(t22, a, fma(t11, dd, -fma(t12, c2, t21 * b2)));
      o.dm0 = fma(a, dd, -b2 * c2);
    }
    if (has1) {
      const double a = __ldcg(e11 + l1), b2 = __ldcg(e12 + l1), c2 = __ldcg(e21 + l1), dd = __ldcg(e22 + l1);
      o.e1 = fma(t22, a, fma(t11, dd, -fma(t12, c2, t21 * b2)));
      o.dm1 = fma(a, dd, -b2 * c2);
    }
  }
}

// ---------------------------------------------------------------------------------
// The accelerated route (F.6-F.9): only the reference determinant of each spin is eliminated; every
// other determinant comes from tables.  With B_l = d_l A (dense: every row depends on every coordinate l through the
// Jacobian J of the backflow map) the paper's tables are, per spin,
//   T = A0^-1 Av,   M_l = A0^-1 B_l,v - A0^-1 B_l,0 T  (F.7),   Y_l = A0^-1 B_l,0 M_l  (F.9),
// and here (derivation pinned on random matrices by the P14b test of the CPU suite):
//   rho = A0^-1,  W0^a = V0^a rho,  m^a = Vv^a - V0^a T   (V^a = d_a phi rows),
//   E[q][p][l] = M_l[p][q] = sum_i rho[p][i] sum_a J_il^a m^a[i][q]     (42-vectors, kept in a per-warp global scratch)
//   Y2[q][p]   = sum_l Y_l[p][q] = sum_i rho[p][i] sum_{i',a'} (sum_a C_ii'^{aa'} W0^a[i][i']) m^{a'}[i'][q]
//   t0_l = sum_i sum_a J_il^a W0^a[i][i],   s0 = sum_{ii'} C_ii' : W0[i][i'] (x) W0[i'][i],   E2_0 = |t0|^2 - s0^up - s0^dn
// and per determinant (substitution blocks T_PQ, k <= 2 per spin), division-free:
//   R = det T_PQ,  e~_l = Tr(adj(T_PQ) E_PQ,l),  b = 2 sum_l det(E_PQ,l) [k = 2] - 2 Tr(adj(T_PQ) Y2_PQ)
//   R^up R^dn E2_X = R^up R^dn E2_0 + 2 R^dn t0.e~^up + 2 R^up t0.e~^dn + 2 e~^up.e~^dn + R^dn b^up + R^up b^dn
// so that  -1/2 lap Psi / Psi = -1/2 (lap J + |grad J|^2) + [ den (t^up + t^dn) + num1 - 1/2 sum_n d_n R R E2_n ] / den
// with den, num1 the first-order sums of the plain path (combined operator B of bf_build).  One walker per warp; lane l
// accumulates the l-dependent part over all determinants, one warp reduction at the end.  Walkers whose reference is
// nearly singular (kappa / (Sigma/D0) criteria of section 5.6) are listed for the explicit kernel.
// ---------------------------------------------------------------------------------
template <int NS, int NMO, int WPB, bool DERIV = false, bool MB = false>
__global__ void __launch_bounds__(WPB * 32, 1)
    backflow_tables_kernel(const __grid_constant__ SysParams P, const WalkerIO io, const BfDet *__restrict__ dets,
                           const BfClasses cls, double *__restrict__ escratch) {
  extern __shared__ __align__(16) unsigned char smem[];
  using BG = BfGeoT<NS, NMO>;
  double *sCf = reinterpret_cast<double *>(smem);
  const int nC = P.c_doubles;
  for (int i = threadIdx.x; i < nC; i += blockDim.x) sCf[i] = P.C[i];
  double *sExp = sCf + nC;
  for (int i = threadIdx.x; i < kExpTab + kRngTab; i += blockDim.x) sExp[i] = P.exp_tab[i];
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double *ws = reinterpret_cast<double *>(smem + P.smem_const_bytes) + warp * BG::total;
  const double *sCd = ws + BG::oCd, *sMO = ws + BG::oMO, *sP = ws + BG::oP, *sS = ws + BG::oS;
  double *sTab = ws + BG::oTab, *sSc = ws + BG::oSc;
  const int wpb = (int)(blockDim.x >> 5);  // warps launched per block (<= WPB)
  double *E = escratch + ((int64_t)blockIdx.x * wpb + warp) * BG::eDoubles;
  const int n_up = P.n_up, n_dn = P.n_dn, ne = P.n_e, nc = 3 * ne;
  constexpr int LS = BG::LS;
  // regions of one spin's tables
  auto tabT = [&](int sp) { return sTab + sp * BG::tSpin; };
  auto tabM1 = [&](int sp) { return sTab + sp * BG::tSpin + NS * 8; };
  auto tabRho = [&](int sp) { return sTab + sp * BG::tSpin + 2 * NS * 8; };
  auto tabG = [&](int sp) { return sTab + sp * BG::tSpin + 3 * NS * 8; };
  auto tabW0 = [&](int sp) { return sTab + sp * BG::tSpin + 4 * NS * 8; };
  auto tabMq = [&](int sp) { return sTab + sp * BG::tSpin + 4 * NS * 8 + 3 * NS * 8; };
  auto tabY2 = [&](int sp) { return sTab + sp * BG::tSpin + 4 * NS * 8 + 6 * NS * 8; };
  for (int64_t w = (int64_t)blockIdx.x * wpb + warp; w < io.M; w += (int64_t)gridDim.x * wpb) {
    double Js, es;
    bf_build<NS, NMO, BG, DERIV, MB>(P, sCf, sExp, ws, io, w, lane, Js, es);
    // ---- reference elimination: [A0 | Av | B0 | Bv | 1], lanes 0-7 spin up, 8-15 spin down (lane c = column c)
    const int c = lane & 7, sp = (lane >> 3) & 1;
    const int ns = sp ? n_dn : n_up, nv = P.nv[sp], e0 = sp ? n_up : 0;
    double detv = 1.0, t0v = 0.0, kap = 0.0;
    {
      double a0[NS], av[NS], b0[NS], bv[NS], ai[NS];
      const bool cA = c < ns, cV = c < nv;
      const int colA = cA ? P.ref_col[sp][c] : 0, colV = cV ? P.virt_col[sp][c] : 0;
#pragma unroll
      for (int q = 0; q < NS; ++q) {
        const bool rq = q < ns;
        const int row = e0 + (rq ? q : 0);
        a0[q] = (rq && cA) ? sMO[(0 * BG::NE + row) * NMO + colA] : ((q == c) ? 1.0 : 0.0);
        av[q] = (rq && cV) ? sMO[(0 * BG::NE + row) * NMO + colV] : 0.0;
        b0[q] = (rq && cA) ? sMO[(1 * BG::NE + row) * NMO + colA] : 0.0;
        bv[q] = (rq && cV) ? sMO[(1 * BG::NE + row) * NMO + colV] : 0.0;
        ai[q] = (rq && cA && q == c) ? 1.0 : 0.0;
      }
      int perm[NS];
      int myrow = 0;
      bool used = !(c < NS);
      const int gbase = lane - c;
#pragma unroll
      for (int k = 0; k < NS; ++k) {
        unsigned key = used ? 0u : (((unsigned)(__double2hiint(a0[k]) & 0x7fffffff) & ~7u) | (unsigned)c);
#pragma unroll
        for (int mm = 1; mm < 8; mm <<= 1) key = max(key, __shfl_xor_sync(0xffffffffu, key, mm));
        const int pl = (int)(key & 7u);
        perm[k] = pl;
        if (c == pl) { used = true; myrow = k; }
        double f[NS];
#pragma unroll
        for (int q = 0; q < NS; ++q) f[q] = __shfl_sync(0xffffffffu, a0[q], gbase + pl);
        const double piv = f[k], inv = 1.0 / piv;
        detv *= piv;
#define QMC_BF_ELIM(v)                                                  \
        {                                                               \
          const double t = v[k] * inv;                                  \
          v[k] = t;                                                     \
          _Pragma("unroll") for (int q = 0; q < NS; ++q) if (q != k) v[q] = fma(-f[q], t, v[q]); \
        }
        QMC_BF_ELIM(a0) QMC_BF_ELIM(av) QMC_BF_ELIM(b0) QMC_BF_ELIM(bv) QMC_BF_ELIM(ai)
#undef QMC_BF_ELIM
      }
      int inversions = 0;
#pragma unroll
      for (int k = 0; k < NS; ++k)
#pragma unroll
        for (int k2 = k + 1; k2 < NS; ++k2) inversions += (perm[k] > perm[k2]) ? 1 : 0;
      if (inversions & 1) detv = -detv;
#pragma unroll
      for (int q = 0; q < NS; ++q) if (q == myrow && c < NS) t0v = b0[q];
#pragma unroll
      for (int mm = 1; mm < 8; mm <<= 1) t0v += shfl_xor_d(t0v, mm);
      unsigned kk = 0u;
#pragma unroll
      for (int k = 0; k < NS; ++k) kk = max(kk, (unsigned)(__double2hiint(av[k]) & 0x7fffffff));
#pragma unroll
      for (int mm = 1; mm < 8; mm <<= 1) kk = max(kk, __shfl_xor_sync(0xffffffffu, kk, mm));
      kap = __hiloint2double((int)min(kk, 0x7ff00000u), 0);
      if (lane < 16) {  // rows in position order: row k of the reduced blocks belongs to position perm[k]
        double *T = tabT(sp), *H = tabM1(sp), *Rho = tabRho(sp), *G = tabG(sp);
#pragma unroll
        for (int k = 0; k < NS; ++k) {
          T[perm[k] * 8 + c] = av[k];
          H[perm[k] * 8 + c] = bv[k];    // A0^-1 Bv for now
          Rho[perm[k] * 8 + c] = ai[k];  // A0^-1[position][electron c]
          G[perm[k] * 8 + c] = b0[k];    // (A0^-1 B0)[position][position c]
        }
      }
    }
    __syncwarp();
    // ---- first-order table M1 = A0^-1 Bv - (A0^-1 B0) T (F.7 for the combined operator), lane c = virtual q
    if (lane < 16 && c < nv) {
      double *T = tabT(sp), *M1 = tabM1(sp), *G = tabG(sp);
      for (int p2 = 0; p2 < ns; ++p2) {
        double t = M1[p2 * 8 + c];
        for (int j = 0; j < ns; ++j) t = fma(-G[p2 * 8 + j], T[j * 8 + c], t);
        M1[p2 * 8 + c] = t;
      }
    }
    // ---- W0^a = V0^a rho (lane c = electron i'), m^a = Vv^a - V0^a T (lane c = virtual q)
    if (lane < 16) {
      const double *T = tabT(sp), *Rho = tabRho(sp);
      double *W0 = tabW0(sp), *Mq = tabMq(sp);
      for (int a = 0; a < 3; ++a)
        for (int i = 0; i < ns; ++i) {
          const double *vrow = sMO + ((2 + a) * BG::NE + e0 + i) * NMO;
          double tw = 0.0, tm = (c < nv) ? vrow[P.virt_col[sp][c < kMaxVirt ? c : 0]] : 0.0;
          for (int k = 0; k < ns; ++k) {
            const double v = vrow[P.ref_col[sp][k]];
            tw = fma(v, Rho[k * 8 + c], tw);
            tm = fma(-v, T[k * 8 + c], tm);
          }
          W0[(a * NS + i) * 8 + c] = (c < ns) ? tw : 0.0;
          Mq[(a * NS + i) * 8 + c] = (c < nv) ? tm : 0.0;
        }
    }
    __syncwarp();
    if (DERIV) {
      // the backflow weight as a parameter (eq. 6 factor): d_w A[i][k] = grad phi_k(rt_i) . pw_i, pw_i = d rt_i / d w (left in
      // the grad J region by bf_build) is one more one-body operator: t_w = sum_i pw_i . W0[i][i] and its first-order table
      // M_w[p][q] = sum_i rho[p][i] pw_i . m[i][q] (F.7), kept where G = A0^-1 B0 was (dead since M1)
      const double *sPw = ws + BG::oGJ;
      double twv = 0.0;
      if (lane < 16) {
        const double *W0 = tabW0(sp), *Mq = tabMq(sp), *Rho = tabRho(sp);
        double *Mw = tabG(sp);
        if (c < ns) twv = fma(sPw[e0 + c], W0[(0 * NS + c) * 8 + c], fma(sPw[32 + e0 + c], W0[(1 * NS + c) * 8 + c], sPw[64 + e0 + c] * W0[(2 * NS + c) * 8 + c]));
        if (c < nv) {
          double f[NS];
#pragma unroll
          for (int i = 0; i < NS; ++i)
            f[i] = (i < ns) ? fma(sPw[e0 + i], Mq[(0 * NS + i) * 8 + c], fma(sPw[32 + e0 + i], Mq[(1 * NS + i) * 8 + c], sPw[64 + e0 + i] * Mq[(2 * NS + i) * 8 + c])) : 0.0;
          for (int p2 = 0; p2 < ns; ++p2) {
            double t = 0.0;
#pragma unroll
            for (int i = 0; i < NS; ++i)
              if (i < ns) t = fma(Rho[p2 * 8 + i], f[i], t);
            Mw[p2 * 8 + c] = t;
          }
        }
      }
#pragma unroll
      for (int mm = 1; mm < 8; mm <<= 1) twv += shfl_xor_d(twv, mm);
      if (c == 0 && lane < 16) sSc[8 + sp] = twv;
    }
    // column b of the (symmetric) Jacobian block J_im = d rt_i / d r_m:  1 + S_i (m = i),  -P_im (m != i)
    auto jcol = [&](int i, int m, int b, double &j0, double &j1, double &j2) {
      double xx, yy, zz, xy, yz, zx;
      if (i == m) {
        xx = 1.0 + sS[i]; yy = 1.0 + sS[32 + i]; zz = 1.0 + sS[64 + i]; xy = sS[96 + i]; yz = sS[128 + i]; zx = sS[160 + i];
      } else {
        const double *pp = sP + BG::pofs(i, m, ne);
        xx = -pp[0]; yy = -pp[1]; zz = -pp[2]; xy = -pp[3]; yz = -pp[4]; zx = -pp[5];
      }
      j0 = (b == 0) ? xx : ((b == 1) ? xy : zx);
      j1 = (b == 0) ? xy : ((b == 1) ? yy : yz);
      j2 = (b == 0) ? zx : ((b == 1) ? yz : zz);
    };
    // ---- t0_l and the E vectors, lane = coordinate l = 3 m + b (two rounds)
    double t0l[2] = {0.0, 0.0};
    for (int rd = 0; rd < 2; ++rd) {
      const int l = lane + 32 * rd;
      if (l < nc) {
        const int m = l / 3, b = l - 3 * m;
        double t = 0.0;
        for (int s2 = 0; s2 < 2; ++s2) {
          const int ns2 = s2 ? n_dn : n_up, nv2 = P.nv[s2], f0 = s2 ? n_up : 0;
          const double *W0 = tabW0(s2), *Mq = tabMq(s2), *Rho = tabRho(s2);
          double jc[NS][3];
#pragma unroll
          for (int i = 0; i < NS; ++i) {
            jc[i][0] = jc[i][1] = jc[i][2] = 0.0;
            if (i < ns2) {
              jcol(f0 + i, m, b, jc[i][0], jc[i][1], jc[i][2]);
              t = fma(jc[i][0], W0[(0 * NS + i) * 8 + i], fma(jc[i][1], W0[(1 * NS + i) * 8 + i], fma(jc[i][2], W0[(2 * NS + i) * 8 + i], t)));
            }
          }
          for (int q = 0; q < nv2; ++q) {
            double acc[NS];
#pragma unroll
            for (int p2 = 0; p2 < NS; ++p2) acc[p2] = 0.0;
#pragma unroll
            for (int i = 0; i < NS; ++i) {
              if (i < ns2) {
                const double f = fma(jc[i][0], Mq[(0 * NS + i) * 8 + q], fma(jc[i][1], Mq[(1 * NS + i) * 8 + q], jc[i][2] * Mq[(2 * NS + i) * 8 + q]));
#pragma unroll
                for (int p2 = 0; p2 < NS; ++p2) acc[p2] = fma(Rho[p2 * 8 + i], f, acc[p2]);
              }
            }
#pragma unroll
            for (int p2 = 0; p2 < NS; ++p2)
              if (p2 < ns2) __stcg(E + ((s2 * kMaxVirt + q) * NS + p2) * LS + l, acc[p2]);
          }
        }
        t0l[rd] = t;
      }
    }
    // ---- R^{a'}[i][i'] = sum_a C_ii'^{aa'} W0^a[i][i'] and s0 = sum R^{a'}[i][i'] W0^{a'}[i'][i], same-spin (i, i') only:
    // one lane per unordered pair forms C_ii' = -J_ii P_ii' - P_ii' J_i'i' + sum_{m != i, i'} P_im P_i'm once and serves
    // both orders (C_i'i is its transpose); lanes 0-15 the diagonal (C_ii from bf_build).  Then Y2[q][p] (lane c = q).
    double *sR = ws + BG::oMO;  // the MO planes are dead
    double s0u = 0.0, s0d = 0.0;
    {
      const int npu = n_up * (n_up - 1) / 2, npd = n_dn * (n_dn - 1) / 2;
      for (int pi = lane; pi < npu + npd; pi += 32) {
        const int s2 = pi >= npu ? 1 : 0;
        int rem = pi - (s2 ? npu : 0);
        const int ns2 = s2 ? n_dn : n_up, f0 = s2 ? n_up : 0;
        int i = 0;
        while (rem >= ns2 - 1 - i) { rem -= ns2 - 1 - i; ++i; }
        const int i2 = i + 1 + rem;  // i < i2 < ns2 (positions within the spin)
        const int gi = f0 + i, gi2 = f0 + i2;
        double cc[9];
        bf_pair_block<BG>(sP, sS, gi, gi2, ne, cc);
        const double *W0 = tabW0(s2);
        const double a0 = W0[(0 * NS + i) * 8 + i2], a1 = W0[(1 * NS + i) * 8 + i2], a2v = W0[(2 * NS + i) * 8 + i2];  // W0^a[i][i2]
        const double b0 = W0[(0 * NS + i2) * 8 + i], b1 = W0[(1 * NS + i2) * 8 + i], b2v = W0[(2 * NS + i2) * 8 + i];  // W0^a[i2][i]
        double acc = 0.0;
#pragma unroll
        for (int a2 = 0; a2 < 3; ++a2) {
          const double r12 = fma(cc[0 + a2], a0, fma(cc[3 + a2], a1, cc[6 + a2] * a2v));            // R^{a2}[i][i2]
          const double r21 = fma(cc[3 * a2 + 0], b0, fma(cc[3 * a2 + 1], b1, cc[3 * a2 + 2] * b2v));  // R^{a2}[i2][i]
          sR[((s2 * 3 + a2) * NS + i) * 8 + i2] = r12;
          sR[((s2 * 3 + a2) * NS + i2) * 8 + i] = r21;
          const double wb = (a2 == 0) ? b0 : ((a2 == 1) ? b1 : b2v), wa = (a2 == 0) ? a0 : ((a2 == 1) ? a1 : a2v);
          acc = fma(r12, wb, fma(r21, wa, acc));
        }
        if (s2) s0d += acc; else s0u += acc;
      }
      if (lane < 16 && c < ns) {
        const int gi = e0 + c;
        const double *W0 = tabW0(sp);
        const double w0 = W0[(0 * NS + c) * 8 + c], w1 = W0[(1 * NS + c) * 8 + c], w2 = W0[(2 * NS + c) * 8 + c];
        const double cxx = sCd[gi], cyy = sCd[32 + gi], czz = sCd[64 + gi], cxy = sCd[96 + gi], cyz = sCd[128 + gi], czx = sCd[160 + gi];
        const double r0 = fma(cxx, w0, fma(cxy, w1, czx * w2)), r1 = fma(cxy, w0, fma(cyy, w1, cyz * w2)),
                     r2 = fma(czx, w0, fma(cyz, w1, czz * w2));
        sR[((sp * 3 + 0) * NS + c) * 8 + c] = r0;
        sR[((sp * 3 + 1) * NS + c) * 8 + c] = r1;
        sR[((sp * 3 + 2) * NS + c) * 8 + c] = r2;
        const double acc = fma(r0, w0, fma(r1, w1, r2 * w2));
        if (sp) s0d += acc; else s0u += acc;
      }
    }
#pragma unroll
    for (int mm = 16; mm > 0; mm >>= 1) {
      s0u += shfl_xor_d(s0u, mm);
      s0d += shfl_xor_d(s0d, mm);
    }
    const double s0v = sp ? s0d : s0u;
    __syncwarp();
    if (lane < 16 && c < nv) {
      const double *Mq = tabMq(sp), *Rho = tabRho(sp);
      double *Y2 = tabY2(sp);
      double S2[NS];
#pragma unroll
      for (int i = 0; i < NS; ++i) {
        S2[i] = 0.0;
        if (i < ns) {
          double t = 0.0;
          for (int i2 = 0; i2 < ns; ++i2)
#pragma unroll
            for (int a2 = 0; a2 < 3; ++a2) t = fma(sR[((sp * 3 + a2) * NS + i) * 8 + i2], Mq[(a2 * NS + i2) * 8 + c], t);
          S2[i] = t;
        }
      }
      for (int p2 = 0; p2 < ns; ++p2) {
        double t = 0.0;
#pragma unroll
        for (int i = 0; i < NS; ++i)
          if (i < ns) t = fma(Rho[p2 * 8 + i], S2[i], t);
        Y2[c * 8 + p2] = t;
      }
    }
    if (c == 0 && lane < 16) {
      sSc[sp * 4 + 0] = detv;
      sSc[sp * 4 + 1] = t0v;
      sSc[sp * 4 + 2] = s0v;
      sSc[sp * 4 + 3] = kap;
    }
    __syncwarp();
    // ---- CI sum over the determinants: uniform scalars in every lane, the l-dependent part per lane.  The records are
    // sorted by class (k_up, k_dn) at setup: one loop per class, the substitution orders known at compile time.
    {
      const double *Tu = tabT(0), *Td = tabT(1), *M1u = tabM1(0), *M1d = tabM1(1), *Y2u = tabY2(0), *Y2d = tabY2(1);
      double den = 0.0, num1 = 0.0, uni = 0.0, accl = 0.0, numw = 0.0;
      const double *Mwu = tabG(0), *Mwd = tabG(1);
      const int nj = kJastrowParams + 7 * P.n_een;
      double *orow = (DERIV && io.O) ? io.O + w * (int64_t)(nj + P.n_det_all + 1) : nullptr;
      const int l0 = lane, l1 = lane + 32;
      const bool has1 = l1 < nc, has0 = l0 < nc;
      const uint2 *raw = reinterpret_cast<const uint2 *>(dets);
      const double *Eu = E, *Ed = E + (int64_t)kMaxVirt * NS * LS;
      auto run_class = [&](auto KU, auto KD, int n_begin, int n_end) {
        constexpr int ku = decltype(KU)::value, kd = decltype(KD)::value;
        if (n_begin >= n_end) return;
        uint2 nx0 = __ldg(raw + 3 * n_begin), nx1 = __ldg(raw + 3 * n_begin + 1), nx2 = __ldg(raw + 3 * n_begin + 2);
        for (int n = n_begin; n < n_end; ++n) {
          const uint2 w0 = nx0, w1 = nx1, w2 = nx2;
          if (n + 1 < n_end) {  // the next record while this one is processed
            nx0 = __ldg(raw + 3 * (n + 1)); nx1 = __ldg(raw + 3 * (n + 1) + 1); nx2 = __ldg(raw + 3 * (n + 1) + 2);
          }
          const double d = __hiloint2double((int)w0.y, (int)w0.x);
          // bytes: k[0] k[1] | p[0][0] p[0][1] p[1][0] p[1][1] q[0][0] q[0][1] | q[1][0] q[1][1] pad...
          BfSpinTerms up, dn;
          bf_spin_terms<ku, NS, LS, DERIV>(Tu, M1u, Y2u, Eu, (w1.x >> 16) & 255u, w1.x >> 24, (w1.y >> 16) & 255u, w1.y >> 24, has0, has1, l0, l1, up, Mwu);
          bf_spin_terms<kd, NS, LS, DERIV>(Td, M1d, Y2d, Ed, w1.y & 255u, (w1.y >> 8) & 255u, w2.x & 255u, (w2.x >> 8) & 255u, has0, has1, l0, l1, dn, Mwd);
          if (DERIV) {
            numw = fma(d, fma(up.Rw, dn.R, up.R * dn.Rw), numw);
            if (orow && lane == 0) orow[nj + (w2.x >> 16)] = up.R * dn.R;  // D_n / D_0, divided by Sigma / D_0 below
          }
          den = fma(d * up.R, dn.R, den);                                      // eq. 4
          num1 = fma(d, fma(up.Rd, dn.R, up.R * dn.Rd), num1);                 // F.6 (first order)
          uni = fma(-2.0 * d, fma(dn.R, up.trY, up.R * dn.trY), uni);          // F.9 (summed over l)
          const double x0 = fma(t0l[0], fma(dn.R, up.e0, up.R * dn.e0), fma(up.e0, dn.e0, fma(dn.R, up.dm0, up.R * dn.dm0)));
          const double x1 = fma(t0l[1], fma(dn.R, up.e1, up.R * dn.e1), fma(up.e1, dn.e1, fma(dn.R, up.dm1, up.R * dn.dm1)));
          accl = fma(2.0 * d, x0 + x1, accl);
        }
      };
      using I0 = std::integral_constant<int, 0>;
      using I1 = std::integral_constant<int, 1>;
      using I2 = std::integral_constant<int, 2>;
      run_class(I0{}, I0{}, cls.start[0], cls.start[1]);
      run_class(I0{}, I1{}, cls.start[1], cls.start[2]);
      run_class(I0{}, I2{}, cls.start[2], cls.start[3]);
      run_class(I1{}, I0{}, cls.start[3], cls.start[4]);
      run_class(I1{}, I1{}, cls.start[4], cls.start[5]);
      run_class(I1{}, I2{}, cls.start[5], cls.start[6]);
      run_class(I2{}, I0{}, cls.start[6], cls.start[7]);
      run_class(I2{}, I1{}, cls.start[7], cls.start[8]);
      run_class(I2{}, I2{}, cls.start[8], cls.start[9]);
      double tt = fma(t0l[0], t0l[0], t0l[1] * t0l[1]);
#pragma unroll
      for (int mm = 16; mm > 0; mm >>= 1) {
        accl += shfl_xor_d(accl, mm);
        tt += shfl_xor_d(tt, mm);
        Js += shfl_xor_d(Js, mm);
        es += shfl_xor_d(es, mm);
      }
      if (lane == 0) {
        const double du = sSc[0], dd = sSc[4];
        const double second = fma(den, tt - sSc[2] - sSc[6], uni + accl);
        const double numt = fma(den, sSc[1] + sSc[5], num1) - 0.5 * second;
        const double sig = du * dd * den;
        const double eloc = es + numt / den + P.vnn;
        if (io.logpsi) io.logpsi[w] = Js + log(fabs(du)) + log(fabs(dd)) + log(fabs(den));
        if (io.sign) io.sign[w] = (sig > 0.0) ? 1.0 : ((sig < 0.0) ? -1.0 : 0.0);
        if (io.eloc) io.eloc[w] = eloc;
        // nearly singular reference: the explicit kernel re-evaluates the walker (criteria of DESIGN.md section 5.6; the
        // second-order tables amplify by one more power of kappa, hence the lower, unscaled thresholds)
        const double ku2 = sSc[3], kd2 = sSc[7], scale = QMC_BF_FALLBACK_ESCALE ? fmax(1.0, fabs(eloc)) : 1.0;
        const bool ok = (den * den <= fmin(kBfFallbackK * scale, kFallbackCap)) && (ku2 * ku2 <= kBfFallbackKappa * scale) &&
                        (kd2 * kd2 <= kBfFallbackKappa * scale);
        if (!ok && io.fb_list) io.fb_list[atomicAdd(io.fb_count, 1)] = (int)w;
        if (DERIV && orow) orow[nj + P.n_det_all] = sSc[8] + sSc[9] + numw / den;
      }
      if (DERIV && orow) {
        __syncwarp();  // lane 0's ratios are visible to the warp
        const double iden = 1.0 / den;
        for (int n = lane; n < P.n_det_all; n += 32) orow[nj + n] *= iden;
      }
    }
    __syncwarp();
  }
}

}  // namespace qmc
