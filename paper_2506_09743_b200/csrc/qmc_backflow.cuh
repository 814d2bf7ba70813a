// qmc_backflow.cuh -- local energy of a backflow-transformed Slater-Jastrow wavefunction:
//   rt_i = r_i + sum_{j != i} K_BF(r_ij) (r_i - r_j),  K_BF(r) = w / r
// orbitals at rt, Jastrow factor at r.  Every row of a Slater matrix now depends on every electron, so the last two
// terms of F.5 and the cross term of F.4 no longer vanish.  First cut: the explicit route, every
// determinant eliminated on its own, one walker per warp.
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
#include "qmc_device.cuh"

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

template <int NS, int NMO>
struct BfGeo {
  static constexpr int NE = 2 * NS;
  static constexpr int oXYZ = 0;                       // [3][32] electron coordinates
  static constexpr int oGJ = oXYZ + 96;                // [3][32] grad_i J
  static constexpr int oS = oGJ + 96;                  // [6][32] S_i = sum_j P_ij
  static constexpr int oC = oS + 192;                  // [NE][NE][9] C blocks
  static constexpr int oMO = oC + NE * NE * 9;         // [5][NE][NMO] MO rows: value, operator, d_x, d_y, d_z
  static constexpr int oW = oMO + 5 * NE * NMO;        // [4][3][NS][NS] W^a of the four problems in flight
  static constexpr int oPr = oW + 4 * 3 * NS * NS;     // [4][2] {det, trace}
  static constexpr int oP = oPr + 8;                   // [NE][NE][6] pair matrices
  static constexpr int total = (oP + NE * NE * 6 + 1) & ~1;
};

template <int NS, int NMO, int WPB>
__global__ void __launch_bounds__(WPB * 32, 1)
    backflow_energy_kernel(const __grid_constant__ SysParams P, const WalkerIO io) {
  extern __shared__ __align__(16) unsigned char smem[];
  using BG = BfGeo<NS, NMO>;
  constexpr int NT = (NMO + 7) / 8;
  // constants: C fragments and the exp table (the layout of load_constants)
  double *sCf = reinterpret_cast<double *>(smem);
  const int nC = P.c_doubles;
  for (int i = threadIdx.x; i < nC; i += blockDim.x) sCf[i] = P.C[i];
  double *sExp = sCf + nC;
  for (int i = threadIdx.x; i < kExpTab + kRngTab; i += blockDim.x) sExp[i] = P.exp_tab[i];
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double *ws = reinterpret_cast<double *>(smem + P.smem_const_bytes) + warp * BG::total;
  double *sXYZ = ws + BG::oXYZ, *sGJ = ws + BG::oGJ, *sS = ws + BG::oS, *sCb = ws + BG::oC, *sMO = ws + BG::oMO,
         *sW = ws + BG::oW, *sPr = ws + BG::oPr, *sP = ws + BG::oP;
  const int n_up = P.n_up, n_dn = P.n_dn, ne = P.n_e;
  const double bw = P.bf_w;
  const bool act = lane < ne;
  const int i = act ? lane : 0;
  for (int64_t w = (int64_t)blockIdx.x * WPB + warp; w < io.M; w += (int64_t)gridDim.x * WPB) {
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
    double px = 0.0, py = 0.0, pz = 0.0, Lx = 0.0, Ly = 0.0, Lz = 0.0;
    Sym3 S{0, 0, 0, 0, 0, 0}, S2{0, 0, 0, 0, 0, 0};
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
      if (act) {
        double *pp = sP + (i * ne + j) * 6;
        pp[0] = Pm.xx; pp[1] = Pm.yy; pp[2] = Pm.zz; pp[3] = Pm.xy; pp[4] = Pm.yz; pp[5] = Pm.zx;
      }
    }
    for (int at = 0; at < P.n_atoms; ++at) {
      const double dx = x - P.atom[at][0], dy = y - P.atom[at][1], dz = z - P.atom[at][2];
      ven = fma(-P.atom[at][3], rsqrt_fast(fma(dx, dx, fma(dy, dy, dz * dz))), ven);
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
      const double *pp = sP + (i * ne + m) * 6;
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
    if (act) {
      double *cb = sCb + (i * ne + i) * 9;
      cb[0] = Cd.xx; cb[1] = Cd.xy; cb[2] = Cd.zx; cb[3] = Cd.xy; cb[4] = Cd.yy; cb[5] = Cd.yz; cb[6] = Cd.zx; cb[7] = Cd.yz; cb[8] = Cd.zz;
      for (int i2 = 0; i2 < ne; ++i2) {
        if (i2 == i) continue;
        const double *pq = sP + (i * ne + i2) * 6;
        const Sym3 Pq{pq[0], pq[1], pq[2], pq[3], pq[4], pq[5]};
        const Sym3 J2{1.0 + sS[i2], 1.0 + sS[32 + i2], 1.0 + sS[64 + i2], sS[96 + i2], sS[128 + i2], sS[160 + i2]};
        double acc[9], t[9];
        sym_mul(Ji, Pq, acc);
        sym_mul(Pq, J2, t);
#pragma unroll
        for (int k = 0; k < 9; ++k) acc[k] = -acc[k] - t[k];
        for (int m = 0; m < ne; ++m) {
          if (m == i || m == i2) continue;
          const double *p1 = sP + (i * ne + m) * 6, *p2 = sP + (i2 * ne + m) * 6;
          sym_mul(Sym3{p1[0], p1[1], p1[2], p1[3], p1[4], p1[5]}, Sym3{p2[0], p2[1], p2[2], p2[3], p2[4], p2[5]}, t);
#pragma unroll
          for (int k = 0; k < 9; ++k) acc[k] += t[k];
        }
        double *co = sCb + (i * ne + i2) * 9;
#pragma unroll
        for (int k = 0; k < 9; ++k) co[k] = acc[k];
      }
    }
    __syncwarp();
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
    // ---- phase 3: every determinant on its own, two at a time (four (determinant, spin) problems of 8 lanes)
    const int c = lane & (kBfLP - 1), slot = lane >> 3, gbase = lane - c;
    const int dsel = slot >> 1, sp = slot & 1;
    const int ns = sp ? n_dn : n_up, e0 = sp ? n_up : 0;
    double sig = 0.0, numk = 0.0;
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
      double e2 = 0.0;
      if (ld < ne) {
        const int spi = (ld < n_up) ? 0 : 1, ii = ld - (spi ? n_up : 0);
        const double *Wi = sW + ((dme * 2 + spi) * 3) * NS * NS;
        const double wi[3] = {Wi[(0 * NS + ii) * NS + ii], Wi[(1 * NS + ii) * NS + ii], Wi[(2 * NS + ii) * NS + ii]};
        for (int j = 0; j < ne; ++j) {
          const int spj = (j < n_up) ? 0 : 1, jj = j - (spj ? n_up : 0);
          const double *Wj = sW + ((dme * 2 + spj) * 3) * NS * NS;
          const double *cb = sCb + (ld * ne + j) * 9;
          const double wj[3] = {Wj[(0 * NS + jj) * NS + jj], Wj[(1 * NS + jj) * NS + jj], Wj[(2 * NS + jj) * NS + jj]};
          double t = 0.0;
#pragma unroll
          for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) t = fma(cb[3 * a + b] * wi[a], wj[b], t);
          if (spi == spj) {
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
              for (int b = 0; b < 3; ++b) t = fma(-cb[3 * a + b] * Wi[(a * NS + ii) * NS + jj], Wj[(b * NS + jj) * NS + ii], t);
          }
          e2 += t;
        }
      }
#pragma unroll
      for (int mm = 8; mm > 0; mm >>= 1) e2 += shfl_xor_d(e2, mm);
      if (ld == 0 && (n0 + dme) < P.n_det_all) {
        const double wn = P.det_cols[n0 + dme].d * sPr[(dme * 2) * 2 + 0] * sPr[(dme * 2 + 1) * 2 + 0];
        sig += wn;                                                                            // eq. 4
        numk = fma(wn, sPr[(dme * 2) * 2 + 1] + sPr[(dme * 2 + 1) * 2 + 1] - 0.5 * e2, numk);  // F.2, F.4, F.5
      }
      __syncwarp();
    }
    // ---- assembly (F.1, eq. 1): lanes 0 and 16 hold the sums of the even and odd determinants
    sig += __shfl_xor_sync(0xffffffffu, sig, 16);
    numk += __shfl_xor_sync(0xffffffffu, numk, 16);
    double Js = act ? Jp : 0.0;
    double es = act ? fma(-0.5, lapJ + fma(gJx, gJx, fma(gJy, gJy, gJz * gJz)), vee + ven) : 0.0;
#pragma unroll
    for (int mm = 16; mm > 0; mm >>= 1) { Js += shfl_xor_d(Js, mm); es += shfl_xor_d(es, mm); }
    if (lane == 0) {
      if (io.logpsi) io.logpsi[w] = Js + log(fabs(sig));
      if (io.sign) io.sign[w] = (sig > 0.0) ? 1.0 : ((sig < 0.0) ? -1.0 : 0.0);
      if (io.eloc) io.eloc[w] = es + numk / sig + P.vnn;
    }
    __syncwarp();
  }
}

}  // namespace qmc
