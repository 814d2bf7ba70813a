// qmc_eval.cuh -- the fused per-walker evaluator: STO atomic orbitals -> MO contraction
// -> Pade Jastrow -> per-spin Gauss-Jordan (A0^-1 [Av | B0 | Bv]) -> excitation tables
// -> CI sum -> E_L assembly.  Citations are /root/reference/PAPER.md lines.
#pragma once
#ifndef QMC_CI_UNROLL
#define QMC_CI_UNROLL 1  // unroll factor of the CI class loops; 1 keeps the kernels small (instruction cache): measured
                         // CO E_L 465 -> 457 us, Metropolis 6.25 -> 6.07 ms against the compiler's own choice of 4
#endif
#include "qmc_device.cuh"

namespace qmc {

// Excitation factors of one spin of one determinant relative to the reference, from the tables
//   T = A0^-1 Av,  Mt = A0^-1 Bv - A0^-1 B0 T                      (F.6/F.7)
//   R  = det T[p,q] = D_X / D_0                                     (reading Q8; H.1)
//   Rd = Tr(adj(T[p,q]) Mt[p,q]) = R * Tr((P A0^-1 A_X P)^-1 P M P) (F.6)
// idx packs four uint8 table indices {11, 12, 21, 22}.
// For E_L the two tables are interleaved, entry = {T, Mt} (one 16-byte load per entry).
template <bool EL>
__device__ __forceinline__ void excite_double(uint32_t idx, const double *__restrict__ T, double &R, double &Rd) {
  const int i11 = idx & 255, i12 = (idx >> 8) & 255, i21 = (idx >> 16) & 255, i22 = idx >> 24;
  if (EL) {
    const double2 *TM = reinterpret_cast<const double2 *>(T);
    const double2 a = TM[i11], b = TM[i12], c = TM[i21], d = TM[i22];
    R = fma(a.x, d.x, -b.x * c.x);
    Rd = fma(d.x, a.y, fma(a.x, d.y, -fma(b.x, c.y, c.x * b.y)));
  } else {
    R = fma(T[i11], T[i22], -T[i12] * T[i21]);
    Rd = 0.0;
  }
}

// General substitution order k (> 2): R = det T[p,q]; Rd = Tr(adj(T[p,q]) Mt[p,q]) = sum_j det(T[p,q] with
// column j taken from Mt[p,q]) -- division-free, valid at R = 0.  Rare path: local-memory k x k LU.
static __device__ __noinline__ double small_det(double *a, int k) {
  double det = 1.0;
  for (int c = 0; c < k; ++c) {
    int piv = c;
    double best = fabs(a[c * k + c]);
    for (int r = c + 1; r < k; ++r)
      if (fabs(a[r * k + c]) > best) { best = fabs(a[r * k + c]); piv = r; }
    if (piv != c) {
      for (int j = 0; j < k; ++j) { const double t = a[c * k + j]; a[c * k + j] = a[piv * k + j]; a[piv * k + j] = t; }
      det = -det;
    }
    const double d = a[c * k + c];
    det *= d;
    if (d == 0.0) return 0.0;
    const double inv = 1.0 / d;
    for (int r = c + 1; r < k; ++r) {
      const double f = a[r * k + c] * inv;
      for (int j = c + 1; j < k; ++j) a[r * k + j] = fma(-f, a[c * k + j], a[r * k + j]);
    }
  }
  return det;
}
template <bool EL>
__device__ __noinline__ void excite_general(const GenSpin *g, const double *T, int RS, double *out) {
  const int k = g->k;
  double R = 1.0, Rd = 0.0;
  if (k > 0) {
    double a[kMaxSpin * kMaxSpin], w[kMaxSpin * kMaxSpin];
    for (int i = 0; i < k; ++i)
      for (int j = 0; j < k; ++j) {
        const int idx = g->p[i] * RS + g->q[j];
        a[i * k + j] = EL ? reinterpret_cast<const double2 *>(T)[idx].x : T[idx];
      }
    for (int i = 0; i < k * k; ++i) w[i] = a[i];
    R = small_det(w, k);
    if (EL)
      for (int c = 0; c < k; ++c) {
        for (int i = 0; i < k * k; ++i) w[i] = a[i];
        for (int i = 0; i < k; ++i) w[i * k + c] = reinterpret_cast<const double2 *>(T)[g->p[i] * RS + g->q[c]].y;
        Rd += small_det(w, k);
      }
  }
  out[0] = R;
  out[1] = Rd;
}

// ---------------------------------------------------------------------------------
// Electron-electron-nucleus Jastrow kernel (D.3): eq. 5 sums it over every nucleus and every
// pair once; each pair enters symmetrised, 1/2 [K(r_ai, r_aj, r_ij) + K(r_aj, r_ai, r_ij)] (reading Q22), i.e.
//   J_een = sum_a sum_{i != j} sum_mu c f(r_ai) g(r_aj) h(r_ij)   over ORDERED pairs with c = c_mu / 2 (P.een[mu][0],
// halved by qmc_setup), Pade factors p(r) = a r/(1 + b r).  For the lane's electron i:
// The lane keeps only its own electron's share: of the two ordered pairs (i,j) and (j,i)
//   u  = c (g_j f_i + f_j g_i),  v' = c (g_j f'_i + f_j g'_i),  vL = c (g_j (f''_i + 2f'_i/r_ai) + f_j (g''_i + 2g'_i/r_ai))
//   J share 1/2 u h;  grad_i += v' h e_ai + u h' e_ij;  lap_i += vL h + u (h'' + 2h'/r_ij) + 2 v' h' e_ai.e_ij.
// Out of line in the plain kernels (rare option, keeps the hot kernels small; een_terms), inlined in the backflow
// kernels (a call there costs more in spills than it saves; een_terms_inl).  out = {J share, grad x, y, z, lap}.
// ---------------------------------------------------------------------------------
template <bool EL>
__device__ __forceinline__ void een_terms_inl(const SysParams &P, const double *sXYZ, int base, int ne, int e, double x, double y,
                                              double z, double *out) {
  double Jp = 0.0, gx = 0.0, gy = 0.0, gz = 0.0, lap = 0.0;
  const int n = P.n_een;
  for (int at = 0; at < P.n_atoms; ++at) {
    const double ax = P.atom[at][0], ay = P.atom[at][1], az = P.atom[at][2];
    const double aix = x - ax, aiy = y - ay, aiz = z - az;
    const double rai2 = fma(aix, aix, fma(aiy, aiy, aiz * aiz));
    const double irai = rsqrt_fast(rai2), rai = rai2 * irai;
    // this electron's factors for every term: value, first derivative, p'' + 2 p'/r
    double fi[kMaxEen], f1[kMaxEen], fL[kMaxEen], gi[kMaxEen], g1[kMaxEen], gL[kMaxEen];
#pragma unroll
    for (int mu = 0; mu < kMaxEen; ++mu) {
      if (mu < n) {
        const double *q = P.een[mu];
        const double d1 = rcp_fast(fma(q[2], rai, 1.0)), d2 = rcp_fast(fma(q[4], rai, 1.0));
        fi[mu] = q[1] * rai * d1;
        gi[mu] = q[3] * rai * d2;
        if (EL) {
          f1[mu] = q[1] * d1 * d1;
          g1[mu] = q[3] * d2 * d2;
          fL[mu] = 2.0 * f1[mu] * (irai - q[2] * d1);   // -2 a b D^-3 + 2 a D^-2 / r
          gL[mu] = 2.0 * g1[mu] * (irai - q[4] * d2);
        }
      }
    }
    double ga = 0.0;  // coefficient of e_ai in grad_i, summed over partners and terms
    for (int o = 1; o < ne; ++o) {
      int j = e + o;
      j -= (j >= ne) ? ne : 0;
      const double xj = sXYZ[base + j], yj = sXYZ[32 + base + j], zj = sXYZ[64 + base + j];
      const double ijx = x - xj, ijy = y - yj, ijz = z - zj;
      const double rij2 = fma(ijx, ijx, fma(ijy, ijy, ijz * ijz));
      const double irij = rsqrt_fast(rij2), rij = rij2 * irij;
      const double ajx = xj - ax, ajy = yj - ay, ajz = zj - az;
      const double raj2 = fma(ajx, ajx, fma(ajy, ajy, ajz * ajz));
      const double raj = raj2 * rsqrt_fast(raj2);
      const double cosA = fma(aix, ijx, fma(aiy, ijy, aiz * ijz)) * irai * irij;  // e_ai . e_ij
      double gij = 0.0;  // coefficient of e_ij in grad_i
#pragma unroll
      for (int mu = 0; mu < kMaxEen; ++mu) {
        if (mu < n) {
          const double *q = P.een[mu];
          const double fj = q[1] * raj * rcp_fast(fma(q[2], raj, 1.0));
          const double gj = q[3] * raj * rcp_fast(fma(q[4], raj, 1.0));
          const double dh = rcp_fast(fma(q[6], rij, 1.0));
          const double h = q[5] * rij * dh;
          const double u = q[0] * fma(gj, fi[mu], fj * gi[mu]);
          Jp = fma(0.5 * u, h, Jp);
          if (EL) {
            const double h1 = q[5] * dh * dh;
            const double hL = 2.0 * h1 * (irij - q[6] * dh);
            const double v1 = q[0] * fma(gj, f1[mu], fj * g1[mu]);
            const double vL = q[0] * fma(gj, fL[mu], fj * gL[mu]);
            ga = fma(v1, h, ga);
            gij = fma(u, h1, gij);
            lap += fma(vL, h, fma(u, hL, 2.0 * v1 * h1 * cosA));
          }
        }
      }
      if (EL) {
        const double sc = gij * irij;
        gx = fma(sc, ijx, gx);
        gy = fma(sc, ijy, gy);
        gz = fma(sc, ijz, gz);
      }
    }
    if (EL) {
      const double sc = ga * irai;
      gx = fma(sc, aix, gx);
      gy = fma(sc, aiy, gy);
      gz = fma(sc, aiz, gz);
    }
  }
  out[0] = Jp;
  out[1] = gx;
  out[2] = gy;
  out[3] = gz;
  out[4] = lap;
}
template <bool EL>
__device__ __noinline__ void een_terms(const SysParams &P, const double *sXYZ, int base, int ne, int e, double x, double y,
                                       double z, double *out) {
  een_terms_inl<EL>(P, sXYZ, base, ne, e, x, y, z, out);
}

// Parameter derivatives of the e-e-n kernel (eq. 6 factors of D.3): for the lane's electron i and term mu the sums over
// nuclei a and partners j != i (the ordered pairs that start at i) of d(c f(r_ai) g(r_aj) h(r_ij))/d(c, a_f, b_f, a_g,
// b_g, a_h, b_h), with p = a r/(1 + b r): dp/da = r/(1 + b r) =: P, dp/db = -a r^2/(1 + b r)^2 = -p P.  q0 = c / 2 is the
// weight of an ordered pair (reading Q22), so d/dc carries the 1/2 explicitly.  Out of line.
__device__ __forceinline__ void een_param_terms_inl(const SysParams &P, const double *sXYZ, int base, int ne, int e, double x,
                                                    double y, double z, int mu, double *dq) {
  const double q0 = P.een[mu][0], q1 = P.een[mu][1], q2 = P.een[mu][2], q3 = P.een[mu][3], q4 = P.een[mu][4],
               q5 = P.een[mu][5], q6 = P.een[mu][6];
  double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0, s4 = 0.0, s5 = 0.0, s6 = 0.0;
  for (int at = 0; at < P.n_atoms; ++at) {
    const double ax = P.atom[at][0], ay = P.atom[at][1], az = P.atom[at][2];
    const double aix = x - ax, aiy = y - ay, aiz = z - az;
    const double rai2 = fma(aix, aix, fma(aiy, aiy, aiz * aiz));
    const double rai = rai2 * rsqrt_fast(rai2);
    const double Pf = rai * rcp_fast(fma(q2, rai, 1.0)), f = q1 * Pf, fb = -f * Pf;
    for (int o = 1; o < ne; ++o) {
      int j = e + o;
      j -= (j >= ne) ? ne : 0;
      const double xj = sXYZ[base + j], yj = sXYZ[32 + base + j], zj = sXYZ[64 + base + j];
      const double ijx = x - xj, ijy = y - yj, ijz = z - zj;
      const double rij2 = fma(ijx, ijx, fma(ijy, ijy, ijz * ijz));
      const double rij = rij2 * rsqrt_fast(rij2);
      const double ajx = xj - ax, ajy = yj - ay, ajz = zj - az;
      const double raj2 = fma(ajx, ajx, fma(ajy, ajy, ajz * ajz));
      const double raj = raj2 * rsqrt_fast(raj2);
      const double Pg = raj * rcp_fast(fma(q4, raj, 1.0)), gv = q3 * Pg, gb = -gv * Pg;
      const double Ph = rij * rcp_fast(fma(q6, rij, 1.0)), h = q5 * Ph, hb = -h * Ph;
      const double gh = gv * h, fg = f * gv;
      s0 = fma(f, gh, s0);
      s1 = fma(Pf, gh, s1);
      s2 = fma(fb, gh, s2);
      s3 = fma(f * Pg, h, s3);
      s4 = fma(f * gb, h, s4);
      s5 = fma(fg, Ph, s5);
      s6 = fma(fg, hb, s6);
    }
  }
  dq[0] = 0.5 * s0;
  dq[1] = q0 * s1;
  dq[2] = q0 * s2;
  dq[3] = q0 * s3;
  dq[4] = q0 * s4;
  dq[5] = q0 * s5;
  dq[6] = q0 * s6;
}
static __device__ __noinline__ void een_param_terms(const SysParams &P, const double *sXYZ, int base, int ne, int e, double x,
                                             double y, double z, int mu, double *dq) {
  een_param_terms_inl(P, sXYZ, base, ne, e, x, y, z, mu, dq);
}

// ---------------------------------------------------------------------------------
// Evaluate the G walkers of this warp.  Lane = g * n_e + e holds electron e of walker g
// at (x, y, z).  Results for walker g are left in ws[oRes + 4 g + {0,1,2}] =
// {log|Psi|, sign, E_L} (E_L only if EL).  All 32 lanes must call.
// ---------------------------------------------------------------------------------
// DERIV: also write the logarithmic parameter derivatives of eq. 6 for the G walkers to dv.O.
// EEN: the wavefunction carries the electron-electron-nucleus kernel D.3 (separate instantiations, so that the
// kernels of the common case stay free of the call and its register spills: measured 459 -> 508 us otherwise).
// ORB = 1 (with EXPL): B = I, i.e. every determinant's inverse; Gamma[i][alpha] = sum_n d_n D_n^up D_n^dn A_n^-1[pos_n(alpha)][i]
// is accumulated behind the common scratch (Geo::oGam), for the orbital-parameter derivatives.
// ORB = 3 (with EXPL and EL): [A_n | B_n | I] is eliminated, so that both A_n^-1 and P_n = A_n^-1 B_n are at hand;
// besides Gamma (= d Sigma / d Phi, unnormalised) the second weight matrix of the nuclear energy gradient is accumulated,
//   Gamma2[i][alpha] = sum_n d_n D_n^up D_n^dn (t_n A_n^-1 - A_n^-1 B_n A_n^-1)[pos_n(alpha)][i],  t_n = t_n^up + t_n^dn
// (= d (sum_n w_n t_n) / d Phi at fixed B; the derivative with respect to B is Gamma itself), and grad_i J is left in
// Geo::oGJ for the caller.
// ORB = 2 (table path, values only): the same Gamma from the reference alone: A0^-1 through an identity block of the
// elimination, Y = d den / d T accumulated in the CI pass, Gamma_virt = A0^-T Y / den, Gamma_occ = A0^-T - Gamma_virt T^T.
// the values-only evaluation on its own (log|Psi| kernel, sampler) uses the compact scratch layout
template <bool EL, bool EXPL, int ORB>
constexpr bool kCompact = !EL && !EXPL && ORB == 0;

// BF (values only): the orbitals are evaluated at the backflow coordinates rt_i = r_i + w sum_{j != i} (r_i - r_j)/r_ij
// (PAPER.md:53 with the inverse kernel of PAPER.md:97), the Jastrow factor at r; the determinant algebra is unchanged.
// E_L of a backflow wavefunction has its own kernel (qmc_backflow.cuh).
// FUSE (with DERIV): the rows O[w][:] of the G walkers are left in shared memory behind the evaluator's scratch
// (ws + Geo::total, row stride n_param) instead of going to HBM: the caller reduces them for the eq. 6 estimator.
template <int NS, int NMO, bool EL, bool X, bool EXPL = false, bool DERIV = false, bool EEN = false, int ORB = 0, bool BF = false,
          bool FUSE = false>
__device__ void eval_walkers(const SysParams &P, const double *__restrict__ sExp,
                             const double *__restrict__ sC, const DetRec *__restrict__ sDet,
                             double *__restrict__ ws, double x, double y, double z, int lane,
                             int det0 = 0, int det_step = 1, const DerivOut dv = DerivOut{}) {
  using GE = Geo<NS, NMO>;
  constexpr int LP = GE::LP, PP = GE::PP, TS = GE::TS, RS = GE::RS;
  // X: closed-shell system that matches the instantiation exactly (n_up = n_dn = NS): sizes fold
  const int n_up = X ? NS : P.n_up, n_dn = X ? NS : P.n_dn, ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G;
  const int g = lane / ne, e = lane - g * ne;
  const bool active = lane < G * ne;
  constexpr bool CP = kCompact<EL, EXPL, ORB>;  // values-only evaluation: compact scratch layout (Geo::oPartC ...)
  double *sPhi = ws + GE::oPhi, *sB = ws + GE::oB, *sXYZ = ws + GE::oXYZC(CP), *sPart = ws + GE::oPartC(CP);
  double *sG = ws + GE::oG, *sT = ws + GE::oT, *sProb = ws + GE::oProbC(CP);
  double *sRes = ws + GE::oResC(CP);

  // backflow here only where orbital VALUES suffice: log|Psi| and Gamma = d ln Sigma / d Phi (ORB 1, 2: orbital_derivatives_kernel)
  static_assert(!BF || (!EL && !DERIV && (ORB == 0 ? !EXPL : (ORB == 1 || ORB == 2))), "backflow: values-only evaluation here");
  // ---- publish coordinates for the pair loop
  sXYZ[lane] = x;  // [xyz][lane]: the pair loop reads consecutive lanes
  sXYZ[32 + lane] = y;
  sXYZ[64 + lane] = z;
  __syncwarp();
  double xa = x, ya = y, za = z;  // where the lane's orbitals are evaluated
  if (BF) {
    const int base = (active ? g : 0) * ne;
    double px = 0.0, py = 0.0, pz = 0.0;
    for (int o = 1; o < ne; ++o) {
      int j = e + o;
      j -= (j >= ne) ? ne : 0;
      const double dx = x - sXYZ[base + j], dy = y - sXYZ[32 + base + j], dz = z - sXYZ[64 + base + j];
      const double ri = rsqrt_fast(fma(dx, dx, fma(dy, dy, dz * dz)));
      px = fma(dx, ri, px);
      py = fma(dy, ri, py);
      pz = fma(dz, ri, pz);
    }
    xa = fma(P.bf_w, px, x);
    ya = fma(P.bf_w, py, y);
    za = fma(P.bf_w, pz, z);
  }

  // ---- stage a5: Pade Jastrow (D.1) and e-e repulsion (eq. 1).
  // Every unordered pair is evaluated once: electron e takes the partners e+1 .. e+(ne-1)/2 (cyclic),
  // and for even ne the lower half also takes e+ne/2; the partner's share of the gradient (the
  // opposite vector) travels by shuffle from the lane that computed the pair.
  double Jp = 0.0, gJx = 0.0, gJy = 0.0, gJz = 0.0, lapJ = 0.0, vee = 0.0;
  double dJa_par = 0.0, dJa_anti = 0.0, dJb = 0.0;  // DERIV: this lane's share of dJ/da_par, dJ/da_anti, dJ/db
  {
    const bool up = e < n_up;
    const int base = (active ? g : 0) * ne;
    const int nfull = (ne - 1) >> 1, nofs = ne >> 1, half = ne >> 1;
    constexpr int kPairUnroll = QMC_PAIR_UNROLL;
#pragma unroll kPairUnroll
    for (int o = 1; o <= nofs; ++o) {
      int j = e + o;
      j -= (j >= ne) ? ne : 0;
      const bool take = (o <= nfull) || (e < half);
      const double dx = x - sXYZ[base + j];
      const double dy = y - sXYZ[32 + base + j];
      const double dz = z - sXYZ[64 + base + j];
      const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
      const double ri = rsqrt_fast(r2);
      const double r = r2 * ri;
      double a = ((j < n_up) == up) ? P.a_par : P.a_anti;
      a = take ? a : 0.0;
      const double di = rcp_fast(fma(P.b, r, 1.0));
      const double adi = a * di;
      Jp = fma(adi, r, Jp);  // u = a r / (1 + b r)
      if (DERIV) {
        // D.1: dK/da = r / (1 + b r) for the pair's own a, dK/db = -a r^2 / (1 + b r)^2
        const double rd = take ? r * di : 0.0;
        const bool same = (j < n_up) == up;
        dJa_par += same ? rd : 0.0;
        dJa_anti += same ? 0.0 : rd;
        dJb = fma(-adi * r, rd, dJb);
      }
      if (EL) {
        const double u1 = adi * di;              // u'  = a / (1 + b r)^2
        const double u2 = -2.0 * P.b * u1 * di;  // u'' = -2 a b / (1 + b r)^3
        const double sc = u1 * ri;
        const double cx = sc * dx, cy = sc * dy, cz = sc * dz;
        lapJ += 2.0 * fma(2.0, sc, u2);          // lap_i K + lap_j K = 2 (u'' + 2 u'/r)
        vee += take ? ri : 0.0;
        int src = e - o;
        src += (src < 0) ? ne : 0;
        const int sl = (lane - e + src) & 31;    // lane that computed the pair (src, e)
        gJx += cx - shfl_d(cx, sl, 32);
        gJy += cy - shfl_d(cy, sl, 32);
        gJz += cz - shfl_d(cz, sl, 32);
      }
    }
  }

  // ---- electron-nucleus Jastrow kernel (D.2): K = N / D, N = w0 r + w1 r^2, D = 1 + w2 r,
  //   K' = (N' - w2 K) / D,  K'' = (N'' - 2 w2 K') / D;  grad_i J += K' d / r,  lap_i J += K'' + 2 K'/r.
  // It has to precede the AO stage, whose combined operator uses the complete grad J.
  double dEn0 = 0.0, dEn1 = 0.0, dEn2 = 0.0;  // DERIV: this lane's share of dJ/dw0, dJ/dw1, dJ/dw2 (D.2)
  if (P.has_en || DERIV) {  // the parameter derivatives are defined (and wanted) at w = 0 too
    for (int at = 0; at < P.n_atoms; ++at) {
      const double dx = x - P.atom[at][0], dy = y - P.atom[at][1], dz = z - P.atom[at][2];
      const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
      const double ri = rsqrt_fast(r2);
      const double r = r2 * ri;
      const double di = rcp_fast(fma(P.en_w2, r, 1.0));
      const double K = r * fma(P.en_w1, r, P.en_w0) * di;
      Jp += K;
      if (DERIV) {  // dK/dw0 = r / D, dK/dw1 = r^2 / D, dK/dw2 = -N r / D^2 = -K r / D
        const double rd = r * di;
        dEn0 += rd;
        dEn1 = fma(r, rd, dEn1);
        dEn2 = fma(-K, rd, dEn2);
      }
      if (EL) {
        const double K1 = (fma(2.0 * P.en_w1, r, P.en_w0) - P.en_w2 * K) * di;
        const double K2 = 2.0 * fma(-P.en_w2, K1, P.en_w1) * di;
        const double sc = K1 * ri;
        gJx = fma(sc, dx, gJx);
        gJy = fma(sc, dy, gJy);
        gJz = fma(sc, dz, gJz);
        lapJ += fma(2.0, sc, K2);
      }
    }
  }

  if (EEN) {  // electron-electron-nucleus kernel (D.3); sXYZ still holds the coordinates
    double t[5];
    een_terms<EL>(P, sXYZ, (active ? g : 0) * ne, ne, e, x, y, z, t);
    Jp += t[0];
    if (EL) {
      gJx += t[1];
      gJy += t[2];
      gJz += t[3];
      lapJ += t[4];
    }
  }

  if (ORB == 3 || ORB == 4) {  // grad_i J for the caller (nuclear energy gradient: d B / d R needs it)
    double *sGJ = ws + GE::oGJ;
    sGJ[lane] = gJx;
    sGJ[32 + lane] = gJy;
    sGJ[64 + lane] = gJz;
  }

  // ---- stages a1-a4: STO shells and AO -> MO contraction.
  // For E_L the gradient and Laplacian are folded into ONE operator per AO (stage a6):
  //   b = -1/2 lap(phi) - grad_i J . grad(phi)      (middle and last terms of F.1)
  // The lane evaluates the AOs of its electron and writes them into a [16 AO rows][S] tile; every
  // 16 rows the warp multiplies the tile into the MO accumulators with DMMA m8n8k4
  // (D[row][mo] += A[row][ao] C[ao][mo]; rows = electrons x {value, operator}).
  constexpr int NT = GE::NT;
  constexpr int MT = GE::mTiles(EL);
  constexpr int S = EL ? GE::S2 : GE::S1;
  double ven = 0.0;
  {
    double acc[MT][NT][2];
#pragma unroll
    for (int m = 0; m < MT; ++m)
#pragma unroll
      for (int t = 0; t < NT; ++t) acc[m][t][0] = acc[m][t][1] = 0.0;
    double *const tile = ws;  // overlays the scratch from offset 0 (all dead here except sXYZ, read above)
    __syncwarp();             // every lane is done with sXYZ
    const int fr = lane >> 2, fk = lane & 3;  // fragment row / k of this lane
    const int oo = GE::opCol(lane) - lane;                         // operator column relative to the value column (32 or 36)
    const int mshift = GE::mergeShift(fr);
    double *const tl = tile + lane;                                // this lane's value column of the tile
    // 32-bit shared addresses of the lane's value / operator columns, kept live in registers
    const uint32_t tl32 = opaque_u32((uint32_t)__cvta_generic_to_shared(tl));
    const uint32_t to32 = EL ? opaque_u32(tl32 + 8u * (uint32_t)oo) : 0u;
    const double *const afrag = tile + fk * S + fr;                // A fragments: + 4 ks S + tile column
    const uint32_t exp32 = opaque_u32((uint32_t)__cvta_generic_to_shared(sExp));  // exp_neg's table
    int chunk = 0;
    double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1.0, r = 1.0, ri = 1.0, gd = 0.0, pw = 1.0;
    uint32_t tr = tl32, tro = to32;  // this lane's tile cells of the next AO row (rows follow the record stream)
    // one uniform loop over the record stream [ATOM a][shells of a] ... (every lane reads the same record)
    {
      for (int s = 0; s < P.n_shell; ++s) {
        const ShellRec &sh = P.shells[s];
        const int meta = sh.meta;
        if ((meta & 15) == SH_POW) {   // the shells that follow carry the radial power r^k
          const int k = (meta >> 4) & 3;
          pw = (k == 1) ? r : ((k == 2) ? r2 : r * r2);
          continue;
        }
        if ((meta & 15) == SH_ATOM) {  // new centre: {zeta, c1, c2, kd} = {X, Y, Z, charge}
          pw = 1.0;
          dx = xa - sh.zeta;
          dy = ya - sh.c1;
          dz = za - sh.c2;
          r2 = fma(dx, dx, fma(dy, dy, dz * dz));
          ri = rsqrt_fast(r2);
          r = r2 * ri;
          if (EL) {
            ven = fma(-sh.kd, ri, ven);
            gd = fma(gJx, dx, fma(gJy, dy, gJz * dz)) * ri;  // grad J . d / r
          }
          continue;
        }
        const double gr = exp_neg_s32(-sh.zeta * r, exp32, P.mc) * pw;  // r^k e^{-zeta r}
        double h = 0.0;
        if (EL) {
          // lap(S r^k e^{-zeta r}) = phi * [zeta^2 - 2 zeta (k+l+1)/r + k (k+2l+1)/r^2]
          const double lapfac = fma(fma(sh.c2, ri, -sh.c1), ri, sh.zeta * sh.zeta);
          const double radlog = fma(sh.kd, ri, -sh.zeta);  // g'/g
          h = fma(-0.5, lapfac, -radlog * gd);
        }
        // value into column lane, combined operator into column opCol(lane): every lane stores
#define put(t, phi, bop)                          \
  do {                                            \
    sts_f64<(t) * S * 8>(tr, (phi));              \
    if (EL) sts_f64<(t) * S * 8>(tro, (bop));     \
  } while (0)
        const int kind = meta & 15;
        uint32_t adv = S * 8;  // bytes the row pointers advance by: one row per AO of the record
        if (kind == SH_S) {
          put(0, gr, gr * h);
        } else if (kind == SH_P) {
          put(0, gr * dx, gr * fma(dx, h, -gJx));
          put(1, gr * dy, gr * fma(dy, h, -gJy));
          put(2, gr * dz, gr * fma(dz, h, -gJz));
          adv = 3 * S * 8;
        } else if (kind == SH_D) {
          adv = 5 * S * 8;
          double Sh, gs;
          Sh = dx * dy; gs = fma(gJx, dy, gJy * dx);
          put(0, gr * Sh, gr * fma(Sh, h, -gs));
          Sh = dy * dz; gs = fma(gJy, dz, gJz * dy);
          put(1, gr * Sh, gr * fma(Sh, h, -gs));
          Sh = dz * dx; gs = fma(gJz, dx, gJx * dz);
          put(2, gr * Sh, gr * fma(Sh, h, -gs));
          Sh = fma(dx, dx, -dy * dy); gs = 2.0 * fma(gJx, dx, -gJy * dy);
          put(3, gr * Sh, gr * fma(Sh, h, -gs));
          Sh = fma(2.0 * dz, dz, -fma(dx, dx, dy * dy));
          gs = 2.0 * fma(2.0 * gJz, dz, -fma(gJx, dx, gJy * dy));
          put(4, gr * Sh, gr * fma(Sh, h, -gs));
        } else {  // a lone p or d function (SH_P1, SH_D1)
          const int m = (meta >> 8) & 15;
          double Sh, gs;
          if (kind == SH_P1) {
            Sh = (m == 0) ? dx : ((m == 1) ? dy : dz);
            gs = (m == 0) ? gJx : ((m == 1) ? gJy : gJz);
          } else if (m == 0) { Sh = dx * dy; gs = fma(gJx, dy, gJy * dx); }
          else if (m == 1) { Sh = dy * dz; gs = fma(gJy, dz, gJz * dy); }
          else if (m == 2) { Sh = dz * dx; gs = fma(gJz, dx, gJx * dz); }
          else if (m == 3) { Sh = fma(dx, dx, -dy * dy); gs = 2.0 * fma(gJx, dx, -gJy * dy); }
          else { Sh = fma(2.0 * dz, dz, -fma(dx, dx, dy * dy)); gs = 2.0 * fma(2.0 * gJz, dz, -fma(gJx, dx, gJy * dy)); }
          put(0, gr * Sh, gr * fma(Sh, h, -gs));
        }
#undef put
        tr += adv;
        if (EL) tro += adv;
        const int flush = meta >> 20;
        if (flush) {
          tr = tl32;
          tro = to32;
          // unused rows of the chunk meet zero rows of C, but must themselves be finite
          for (int pr = flush; pr < kChunk; ++pr) {
            tl[pr * S] = 0.0;
            if (EL) tl[pr * S + oo] = 0.0;
          }
          __syncwarp();
          const double *cf = sC + chunk * ((kChunk / 4) * NT * 32) + lane;
#pragma unroll
          for (int ks = 0; ks < kChunk / 4; ++ks) {
            double bf[NT];
#pragma unroll
            for (int t = 0; t < NT; ++t) bf[t] = cf[(ks * NT + t) * 32];
            const double *arow = afrag + 4 * ks * S;
#pragma unroll
            for (int m = 0; m < MT; ++m) {
              const double a = arow[GE::tileCol(EL, m) + ((EL && GE::MERGE && m == GE::VT) ? mshift : 0)];
#pragma unroll
              for (int t = 0; t < NT; ++t) dmma884(acc[m][t][0], acc[m][t][1], a, bf[t]);
            }
          }
          ++chunk;
          __syncwarp();
        }
      }
    }
    // the tile is dead: the MO rows overlay it.  D fragments -> MO rows: the lane holds rows fr of every
    // M-tile, columns 8 t + 2 fk + {0,1}
#pragma unroll
    for (int m = 0; m < MT; ++m) {
      bool isB = false;
      int el = 8 * m + fr;
      if (EL) {
        if (GE::MERGE) {
          if (m == GE::VT) { isB = fr >= 4; el = 8 * GE::VT + (fr & 3); }
          else if (m > GE::VT) { isB = true; el = 8 * (m - GE::VT - 1) + fr; }
        } else if (m >= GE::VTc) { isB = true; el = 8 * (m - GE::VTc) + fr; }
      }
      double *dst = (isB ? sB : sPhi);
      if (el < G * ne) {
#pragma unroll
        for (int t = 0; t < NT; ++t) {
          const int col = 8 * t + 2 * fk;
          if (col < NMO) *reinterpret_cast<double2 *>(dst + GE::moIdx(EL, el, col)) = make_double2(acc[m][t][0], acc[m][t][1]);
        }
      }
    }
    __syncwarp();
  }
  {
    // per-electron scalars: J/2-sum and the electron's share of the energy
    sPart[lane * 2 + 0] = Jp;
    sPart[lane * 2 + 1] = EL ? (fma(-0.5, lapJ + fma(gJx, gJx, fma(gJy, gJy, gJz * gJz)), vee + ven)) : 0.0;
    if (DERIV) {  // the coordinate scratch is dead (and the tile that overlaid it too)
      sXYZ[lane * 3 + 0] = dJa_par;
      sXYZ[lane * 3 + 1] = dJa_anti;
      sXYZ[lane * 3 + 2] = dJb;
    }
  }
  __syncwarp();

  if (EXPL) {
    // ---- explicit path (Fig. 11's "explicit"): every determinant is eliminated on its own,
    // D_n = det A_n, t_n = Tr(A_n^-1 B_n) (G.7 with the combined operator); no excitation tables.
    // Used for walkers whose reference determinant is nearly singular (kFallbackK).
    const int c = lane % LP, slot = lane / LP, gbase = lane - c;
    const int nprob = 2 * G;
    double sig = 0.0, numk = 0.0;
    double *sGam = ws + GE::oGam, *sInv = ws + GE::oInv;
    int *sCol = reinterpret_cast<int *>(ws + GE::oCol);
    double *sGam2 = ws + GE::oGam2, *sStage = ws + GE::oStage, *sX = ws + GE::oX;
    if (ORB == 1 || ORB == 3) {
      for (int i = lane; i < GE::ROWS * NMO; i += 32) {
        sGam[i] = 0.0;
        if (ORB == 3) sGam2[i] = 0.0;
      }
      __syncwarp();
    }
    // this warp takes determinants det0, det0 + det_step, ... (the block shares one walker group)
    DetCols nxt = P.det_cols[det0 < P.n_det_all ? det0 : 0];
    for (int n = det0; n < P.n_det_all; n += det_step) {
      const DetCols dc = nxt;
      if (n + det_step < P.n_det_all) nxt = P.det_cols[n + det_step];  // hide the L2 latency behind the elimination
      for (int pass = 0; pass * PP < nprob; ++pass) {
        const int pr = pass * PP + slot;
        const bool pvalid = pr < nprob;
        const int pg = pvalid ? (pr >> 1) : 0, sp = pr & 1;
        const int ns = sp ? n_dn : n_up, e0 = sp ? n_up : 0;
        double a0[NS], b0[NS];
        double bi[ORB == 3 ? NS : 1];  // ORB = 3: identity block beside B
        {
          const bool cA = c < ns;
          const int colA = cA ? dc.col[sp][c < kMaxSpin ? c : 0] : 0;
#pragma unroll
          for (int i = 0; i < NS; ++i) {
            const int row = pg * ne + e0 + (i < ns ? i : 0);
            const bool ri = i < ns;
            a0[i] = (ri && cA) ? sPhi[GE::moIdx(EL, row, colA)] : ((i == c) ? 1.0 : 0.0);
            if (ORB == 1) b0[i] = (ri && cA && i == c) ? 1.0 : 0.0;  // B = I: the reduced block is A_n^-1 itself
            else b0[i] = (ri && cA) ? sB[EL ? GE::moIdx(EL, row, colA) : 0] : 0.0;
            if (ORB == 3) bi[i] = (ri && cA && i == c) ? 1.0 : 0.0;
          }
        }
        double det = 1.0;
        int perm[NS];
        int myrow = 0;
        bool used = !(c < NS);
#pragma unroll
        for (int k = 0; k < NS; ++k) {
          unsigned key = used ? 0u : (((unsigned)(__double2hiint(a0[k]) & 0x7fffffff) & ~(unsigned)(LP - 1)) | (unsigned)c);
#pragma unroll
          for (int m = 1; m < LP; m <<= 1) key = max(key, __shfl_xor_sync(0xffffffffu, key, m));
          const int pl = (int)(key & (unsigned)(LP - 1));
          perm[k] = pl;
          if (c == pl) { used = true; myrow = k; }
          double f[NS];
#pragma unroll
          for (int i = 0; i < NS; ++i) f[i] = __shfl_sync(0xffffffffu, a0[i], gbase + pl);
          const double piv = f[k];
          const double inv = 1.0 / piv;
          det *= piv;
          double t = a0[k] * inv;
          a0[k] = t;
#pragma unroll
          for (int i = 0; i < NS; ++i) if (i != k) a0[i] = fma(-f[i], t, a0[i]);
          t = b0[k] * inv;
          b0[k] = t;
#pragma unroll
          for (int i = 0; i < NS; ++i) if (i != k) b0[i] = fma(-f[i], t, b0[i]);
          if (ORB == 3) {
            t = bi[k] * inv;
            bi[k] = t;
#pragma unroll
            for (int i = 0; i < NS; ++i) if (i != k) bi[i] = fma(-f[i], t, bi[i]);
          }
        }
        int inversions = 0;
#pragma unroll
        for (int k = 0; k < NS; ++k)
#pragma unroll
          for (int k2 = k + 1; k2 < NS; ++k2) inversions += (perm[k] > perm[k2]) ? 1 : 0;
        if (inversions & 1) det = -det;
        double t0 = 0.0;
#pragma unroll
        for (int i = 0; i < NS; ++i) if (i == myrow && c < NS) t0 = b0[i];
#pragma unroll
        for (int m = 1; m < LP; m <<= 1) t0 += shfl_xor_d(t0, m);
        if (pvalid && c == 0) {
          sProb[pr * 4 + 0] = det;
          sProb[pr * 4 + 2] = t0;
        }
        if ((ORB == 1 || ORB == 3) && pvalid && c < NS) {
          // row k of the reduced block belongs to reference position perm[k]: A_n^-1[perm[k]][electron c]
#pragma unroll
          for (int k = 0; k < NS; ++k) {
            sInv[(pr * NS + k) * NS + c] = (ORB == 3) ? bi[ORB == 3 ? k : 0] : b0[k];
            if (c == 0) sCol[pr * NS + k] = (perm[k] < ns) ? (int)dc.col[sp][perm[k] < kMaxSpin ? perm[k] : 0] : -1;
          }
        }
        if (ORB == 3) {
          // X = P A^-1, P = A^-1 B: lane c holds column c of P (rows in elimination order) and column c (electron c)
          // of A^-1; P is staged so that every lane reads all of it:
          //   X[perm[k']][e] = sum_k P[perm[k']][perm[k]] A^-1[perm[k]][e],  P[perm[k']][perm[k]] = stage[perm[k]][k']
          double *gs = sStage + slot * NS * NS;
          if (c < NS) {
#pragma unroll
            for (int k = 0; k < NS; ++k) gs[c * NS + k] = b0[k];
          }
          __syncwarp();
          double xk[NS];
#pragma unroll
          for (int k2 = 0; k2 < NS; ++k2) xk[k2] = 0.0;
#pragma unroll
          for (int k = 0; k < NS; ++k) {
            const double ak = bi[ORB == 3 ? k : 0];
            const double *gcol = gs + perm[k] * NS;
#pragma unroll
            for (int k2 = 0; k2 < NS; ++k2) xk[k2] = fma(gcol[k2], ak, xk[k2]);
          }
          __syncwarp();
          if (pvalid && c < NS) {
#pragma unroll
            for (int k2 = 0; k2 < NS; ++k2) sX[(pr * NS + k2) * NS + c] = xk[k2];
          }
        }
      }
      __syncwarp();
      if (ORB == 1 || ORB == 3) {
        // d ln D / d A[i][j] = A^-1[j][i], weighted by d_n D_n^up D_n^dn (both determinants are known only now)
        for (int pass = 0; pass * PP < nprob; ++pass) {
          const int pr = pass * PP + slot;
          if (pr < nprob) {
            const int pg = pr >> 1, sp = pr & 1;
            const int ns = sp ? n_dn : n_up, e0 = sp ? n_up : 0;
            const double w = dc.d * sProb[pr * 4 + 0] * sProb[(pr ^ 1) * 4 + 0];
            const double tt = sProb[pr * 4 + 2] + sProb[(pr ^ 1) * 4 + 2];  // t_n = t_n^up + t_n^dn
            if (c < ns) {
              const int row = pg * ne + e0 + c;
#pragma unroll
              for (int k = 0; k < NS; ++k) {
                const int col = sCol[pr * NS + k];
                if (col >= 0) {
                  const double ai = sInv[(pr * NS + k) * NS + c];
                  sGam[row * NMO + col] = fma(w, ai, sGam[row * NMO + col]);
                  if (ORB == 3) sGam2[row * NMO + col] = fma(w, fma(tt, ai, -sX[(pr * NS + k) * NS + c]), sGam2[row * NMO + col]);
                }
              }
            }
          }
        }
      }
      if (lane < G) {
        const double w = dc.d * sProb[(2 * lane) * 4 + 0] * sProb[(2 * lane + 1) * 4 + 0];
        sig += w;                                                                  // eq. 4
        numk = fma(w, sProb[(2 * lane) * 4 + 2] + sProb[(2 * lane + 1) * 4 + 2], numk);  // F.2 / F.4
      }
      __syncwarp();
    }
    if (lane < G) {
      double Jsum = 0.0, esum = 0.0;
      for (int j = 0; j < ne; ++j) {
        Jsum += sPart[(lane * ne + j) * 2 + 0];
        esum += sPart[(lane * ne + j) * 2 + 1];
      }
      // partial sums of this warp's determinants; the kernel combines the warps of the block
      sRes[lane * 4 + 0] = sig;
      sRes[lane * 4 + 1] = numk;
      sRes[lane * 4 + 2] = Jsum;
      sRes[lane * 4 + 3] = esum;
    }
    __syncwarp();
    return;
  }

  // ---- stages a7-a8: per (walker, spin) Gauss-Jordan with partial pivoting on the augmented
  // matrix [A0 | Av | B0 | Bv]; lane c of a group of LP lanes owns column c of every block.
  // Result: T = A0^-1 Av, Gm = A0^-1 B0, H = A0^-1 Bv, det A0.  (F.6/F.7)
  {
    const int c = lane % LP, slot = lane / LP, gbase = lane - c;
    const int nprob = 2 * G;
    for (int pass = 0; pass * PP < nprob; ++pass) {
      const int pr = pass * PP + slot;
      const bool pvalid = pr < nprob;
      const int pg = pvalid ? (pr >> 1) : 0, sp = pr & 1;
      const int ns = sp ? n_dn : n_up, nv = P.nv[sp], e0 = sp ? n_up : 0;
      double a0[NS], av[NS], b0[EL ? NS : 1], bv[EL ? NS : 1];
      constexpr bool INV = (ORB == 2 || ORB == 4);  // identity block -> A0^-1
      double ai[INV ? NS : 1];
      {
        const bool cA = c < ns, cV = c < nv;
        const int colA = cA ? P.ref_col[sp][c < kMaxSpin ? c : 0] : 0;
        const int colV = cV ? P.virt_col[sp][c < kMaxVirt ? c : 0] : 0;
#pragma unroll
        for (int i = 0; i < NS; ++i) {
          const int row = pg * ne + e0 + (i < ns ? i : 0);
          const bool ri = i < ns;
          a0[i] = (ri && cA) ? sPhi[GE::moIdx(EL, row, colA)] : ((i == c) ? 1.0 : 0.0);  // identity padding
          av[i] = (ri && cV) ? sPhi[GE::moIdx(EL, row, colV)] : 0.0;
          if (INV) ai[i] = (ri && cA && i == c) ? 1.0 : 0.0;
          if (EL) {
            b0[i] = (ri && cA) ? sB[GE::moIdx(EL, row, colA)] : 0.0;
            bv[i] = (ri && cV) ? sB[GE::moIdx(EL, row, colV)] : 0.0;
          }
        }
      }
      // Pivoting is by COLUMN: at step k the not-yet-used A0 column with the largest |entry| in row k
      // becomes the pivot; columns live in lanes, so nothing moves.  Row k of the reduced right-hand
      // sides then belongs to reference position perm[k] (the pivot lane).
      double det = 1.0;
      int perm[NS];
      int myrow = 0;
      bool used = !(c < NS);
#pragma unroll
      for (int k = 0; k < NS; ++k) {
        // 32-bit monotone key of |a0[k]| with the lane index in the low bits: unique arg-max
#if QMC_EARLY_INV
        const double myinv = rcp_fast(a0[k]);  // off the critical path: overlaps the arg-max shuffles
#endif
        unsigned key = used ? 0u : (((unsigned)(__double2hiint(a0[k]) & 0x7fffffff) & ~(unsigned)(LP - 1)) | (unsigned)c);
#pragma unroll
        for (int m = 1; m < LP; m <<= 1) key = max(key, __shfl_xor_sync(0xffffffffu, key, m));
        const int pl = (int)(key & (unsigned)(LP - 1));
        perm[k] = pl;
        if (c == pl) { used = true; myrow = k; }
        double f[NS];
#pragma unroll
        for (int i = 0; i < NS; ++i) f[i] = __shfl_sync(0xffffffffu, a0[i], gbase + pl);
        const double piv = f[k];
#if QMC_EARLY_INV
        const double inv = shfl_d(myinv, gbase + pl, 32);
#else
        const double inv = rcp_fast(piv);
#endif
        det *= piv;
        {
          double t = a0[k] * inv;
          a0[k] = t;
#pragma unroll
          for (int i = 0; i < NS; ++i) if (i != k) a0[i] = fma(-f[i], t, a0[i]);
          t = av[k] * inv;
          av[k] = t;
#pragma unroll
          for (int i = 0; i < NS; ++i) if (i != k) av[i] = fma(-f[i], t, av[i]);
          if (INV) {
            t = ai[k] * inv;
            ai[k] = t;
#pragma unroll
            for (int i = 0; i < NS; ++i) if (i != k) ai[i] = fma(-f[i], t, ai[i]);
          }
          if (EL) {
            t = b0[k] * inv;
            b0[k] = t;
#pragma unroll
            for (int i = 0; i < NS; ++i) if (i != k) b0[i] = fma(-f[i], t, b0[i]);
            t = bv[k] * inv;
            bv[k] = t;
#pragma unroll
            for (int i = 0; i < NS; ++i) if (i != k) bv[i] = fma(-f[i], t, bv[i]);
          }
        }
      }
      {  // sign of the permutation k -> perm[k]
        int inversions = 0;
#pragma unroll
        for (int k = 0; k < NS; ++k)
#pragma unroll
          for (int k2 = k + 1; k2 < NS; ++k2) inversions += (perm[k] > perm[k2]) ? 1 : 0;
        if (inversions & 1) det = -det;
      }
      // kappa = max |T[p][q]| of this problem: the conditioning estimate of the explicit-fallback criterion
      // (kFallbackKappa; T = A0^-1 Av blows up like 1/sigma_min(A0) when the reference alone is nearly singular).
      // Arg-max on the high word of |T| (monotone for positive doubles; Inf and NaN of a singular reference sort above
      // every finite value, are clamped to +Inf and so flag the walker): kappa to a relative 2^-20.
      double kap = 0.0;
      if (EL || INV) {
        unsigned kk = 0u;
#pragma unroll
        for (int k = 0; k < NS; ++k) kk = max(kk, (unsigned)(__double2hiint(av[k]) & 0x7fffffff));  // columns c >= nv hold zeros
#pragma unroll
        for (int m = 1; m < LP; m <<= 1) kk = max(kk, __shfl_xor_sync(0xffffffffu, kk, m));
        kap = __hiloint2double((int)min(kk, 0x7ff00000u), 0);  // Inf for every non-finite entry
      }
      // t0 = Tr(A0^-1 B0)   (G.7, applied to the combined operator)
      double t0 = 0.0;
      if (EL) {
#pragma unroll
        for (int i = 0; i < NS; ++i) if (i == myrow && c < NS) t0 = b0[i];
#pragma unroll
        for (int m = 1; m < LP; m <<= 1) t0 += shfl_xor_d(t0, m);
        // Mtab = A0^-1 Bv - (A0^-1 B0) T   (F.7), column c in this lane;
        // rows stay in elimination order (row k <-> position perm[k]) on both sides.
        double *gs = sG + slot * NS * NS;
        if (c < NS) {
#pragma unroll
          for (int i = 0; i < NS; ++i) gs[c * NS + i] = b0[i];  // gs[j][k] = Gm[perm[k]][j]
        }
        if (ORB == 4 && pvalid) {  // keep G = A0^-1 B0 and H = A0^-1 Bv in position order for the adjoint assembly
#pragma unroll
          for (int k = 0; k < NS; ++k) {
            if (c < NS) (ws + GE::oX)[(pr * NS + perm[k]) * NS + c] = b0[k];
            (ws + GE::oH)[(pr * NS + perm[k]) * LP + c] = bv[k];
          }
        }
        __syncwarp();
#pragma unroll
        for (int k = 0; k < NS; ++k) {
          const double tj = av[k];  // T[perm[k]][c]
          const double *gcol = gs + perm[k] * NS;
#pragma unroll
          for (int i = 0; i < NS; ++i) bv[i] = fma(-gcol[i], tj, bv[i]);
        }
        __syncwarp();
      }
      if (pvalid) {
#pragma unroll
        for (int k = 0; k < NS; ++k) {
          if (EL) reinterpret_cast<double2 *>(sT)[pr * TS + perm[k] * RS + c] = make_double2(av[k], bv[EL ? k : 0]);
          else sT[pr * TS + perm[k] * RS + c] = av[k];
          if (INV && c < NS) (ws + GE::oInv)[(pr * NS + perm[k]) * NS + c] = ai[INV ? k : 0];  // A0^-1[position][electron]
        }
        if (c == 0) {
          if (EL) {
            reinterpret_cast<double2 *>(sT)[pr * TS + NS * RS] = make_double2(1.0, 0.0);
            reinterpret_cast<double2 *>(sT)[pr * TS + NS * RS + 1] = make_double2(0.0, 0.0);
          } else {
            sT[pr * TS + NS * RS] = 1.0;
            sT[pr * TS + NS * RS + 1] = 0.0;
          }
          sProb[pr * 4 + 0] = det;  // det A0 of this spin; the logarithm is taken once, of D0^up D0^dn (Sigma / D0)
          sProb[pr * 4 + 2] = t0;
          if (EL || INV) sProb[pr * 4 + 3] = kap;
        }
      }
    }
  }
  __syncwarp();

  // ---- stage a9: CI sum over determinants (eq. 4; F.2/F.4)
  // ---- stage a10: assembly (eq. 1; F.1)
  {
    const int LW = pow2floor(32 / G);
    const int wg = lane / LW, sub = lane - wg * LW;
    const bool wvalid = wg < G;
    const int pu = 2 * (wvalid ? wg : 0), pd = pu + 1;
    const double *Tu = sT + (EL ? 2 : 1) * pu * TS, *Td = sT + (EL ? 2 : 1) * pd * TS;
    double den = (sub == 0) ? P.d_ref : 0.0, num = 0.0;  // determinants equal to the reference: R = 1, Rd = 0
    // table entry at byte offset off8 (in units of 8-byte entries) from the walker's up-spin table
    const char *Tb = reinterpret_cast<const char *>(Tu);
    auto entry = [&](uint32_t off8, double &R, double &D) {
      if (EL) {
        const double2 v = *reinterpret_cast<const double2 *>(Tb + 2 * off8);
        R = v.x;
        D = v.y;
      } else {
        R = *reinterpret_cast<const double *>(Tb + off8);
        D = 0.0;
      }
    };
    constexpr int kCiUnroll = QMC_CI_UNROLL;
    // FUSE: D_n / D_0 of every determinant is kept (kernel order: reference-equal ones, classes 1-4, general) in the
    // walker's shared-memory row; the caller divides by Sigma / D_0 -- no second pass over the determinants
    double *const sRn = ws + GE::total + (wvalid ? wg : 0) * (kJastrowParams + 7 * P.n_een + P.n_det_all) + kJastrowParams +
                        7 * P.n_een + P.n_ref;
    // class 1: one substitution in one spin -- one table entry
#pragma unroll kCiUnroll
    for (int n = sub; n < P.n_a1; n += LW) {
      const DetRec dr = sDet[n];
      double R, D;
      entry(dr.up, R, D);
      den = fma(dr.d, R, den);
      if (EL) num = fma(dr.d, D, num);
      if (FUSE && wvalid) sRn[n] = R;
    }
    // class 2: one substitution in each spin -- two table entries
#pragma unroll kCiUnroll
    for (int n = P.n_a1 + sub; n < P.n_a2; n += LW) {
      const DetRec dr = sDet[n];
      double Ru, Du, Rd, Dd;
      entry(dr.up, Ru, Du);
      entry(dr.dn, Rd, Dd);
      const double w = dr.d * Ru;
      den = fma(w, Rd, den);
      if (EL) num = fma(dr.d, Du * Rd, fma(w, Dd, num));
      if (FUSE && wvalid) sRn[n] = Ru * Rd;
    }
    // class 3: two substitutions in one spin, the other spin as in the reference -- one 2x2 block
#pragma unroll kCiUnroll
    for (int n = P.n_a2 + sub; n < P.n_b; n += LW) {
      const DetRec dr = sDet[n];
      double a, am, b, bm, c, cm, d, dm;
      entry(dr.up & 0xffffu, a, am);
      entry(dr.up >> 16, b, bm);
      entry(dr.dn & 0xffffu, c, cm);
      entry(dr.dn >> 16, d, dm);
      const double R3 = fma(a, d, -b * c);
      den = fma(dr.d, R3, den);
      if (EL) num = fma(dr.d, fma(d, am, fma(a, dm, -fma(b, cm, c * bm))), num);
      if (FUSE && wvalid) sRn[n] = R3;
    }
    // class 4: the rest with at most two per spin -- 2x2 sub-determinants in both spins
#pragma unroll kCiUnroll
    for (int n = P.n_b + sub; n < P.n_det; n += LW) {
      const DetRec dr = sDet[n];
      double Ru, Du, Rd, Dd;
      excite_double<EL>(dr.up, Tu, Ru, Du);
      excite_double<EL>(dr.dn, Td, Rd, Dd);
      const double w = dr.d * Ru;
      den = fma(w, Rd, den);
      if (EL) num = fma(dr.d, Du * Rd, fma(w, Dd, num));
      if (FUSE && wvalid) sRn[n] = Ru * Rd;
    }
    // determinants with more than two substitutions in a spin (general sub-determinants)
    for (int n = sub; n < P.n_gen; n += LW) {
      double u[2], v[2];
      excite_general<EL>(&P.gen[n].s[0], Tu, RS, u);
      excite_general<EL>(&P.gen[n].s[1], Td, RS, v);
      const double dn = P.gen[n].d, w = dn * u[0];
      den = fma(w, v[0], den);
      if (EL) num = fma(dn, u[1] * v[0], fma(w, v[1], num));
      if (FUSE && wvalid) sRn[P.n_det + n] = u[0] * v[0];
    }
    double Jsum = 0.0, esum = 0.0;
    if (wvalid)
      for (int j = sub; j < ne; j += LW) {
        Jsum += sPart[(wg * ne + j) * 2 + 0];
        if (EL) esum += sPart[(wg * ne + j) * 2 + 1];
      }
    for (int m = 1; m < LW; m <<= 1) {
      den += shfl_xor_d(den, m);
      Jsum += shfl_xor_d(Jsum, m);
      if (EL) {
        num += shfl_xor_d(num, m);
        esum += shfl_xor_d(esum, m);
      }
    }
    if (wvalid && sub == 0) {
      // Sigma = D0^up D0^dn (Sigma / D0) (eq. 4): one table-driven logarithm of the product when it and its
      // intermediate are comfortably normal, else the library's, factor by factor (tiny or huge determinants, zeros,
      // NaN).  sign(Sigma) likewise.
      const double du = sProb[pu * 4 + 0], dd = sProb[pd * 4 + 0];
      const double d2 = du * dd, sig = d2 * den;
      const double a2 = fabs(d2), as = fabs(sig);
      double lg, sgn;
      if (a2 > 1e-280 && a2 < 1e280 && as > 1e-280 && as < 1e280) {
        lg = log_pos(as, reinterpret_cast<const double2 *>(sExp + kExpTab), P.mc);
        sgn = (sig > 0.0) ? 1.0 : -1.0;
      } else {
        lg = log(fabs(du)) + log(fabs(dd)) + log(fabs(den));
        const double s1 = (du > 0.0) ? 1.0 : ((du < 0.0) ? -1.0 : 0.0), s2 = (dd > 0.0) ? 1.0 : ((dd < 0.0) ? -1.0 : 0.0);
        sgn = s1 * s2 * ((den > 0.0) ? 1.0 : ((den < 0.0) ? -1.0 : 0.0));
      }
      sRes[wg * 4 + 0] = Jsum + lg;
      sRes[wg * 4 + 1] = sgn;
      if (FUSE) (ws + GE::total)[(G + 2) * (kJastrowParams + 7 * P.n_een + P.n_det_all) + wg] = 1.0 / den;
      const double eloc = EL ? esum + (sProb[pu * 4 + 2] + sProb[pd * 4 + 2]) + num / den + P.vnn : 0.0;
      if (EL) sRes[wg * 4 + 2] = eloc;
      // explicit fallback when the estimated table-path error of E_L exceeds a tenth of the parity bound
      // 1e-8 max(1, |E_L|): ~1e-15 kappa^2 with kappa = max |T| of either spin (a nearly
      // singular reference whatever the size of Sigma) or 1.2e-15 (Sigma/D_0)^2; or when that of log|Psi|,
      // ~1e-15 max(kappa, |Sigma/D_0|), nears a tenth of its absolute bound 1e-10 (the two caps); NaN / Inf flag too
      if (EL) {
        const double ku = sProb[pu * 4 + 3], kd = sProb[pd * 4 + 3];
        const double scale = fmax(1.0, fabs(eloc)), kthr = fmin(kFallbackKappa * scale, kFallbackKappaCap);
        const bool ok = (den * den <= fmin(kFallbackK * scale, kFallbackCap)) && (ku * ku <= kthr) && (kd * kd <= kthr);
        sRes[wg * 4 + 3] = ok ? 0.0 : 1.0;
      }
    }
    if (ORB == 4) {
      // ---- table route of the nuclear energy gradient: the two weight matrices of d_j K, K = F / den,
      //   F = den (t0^up + t0^dn) + num,  d_j K = (d_j F - K d_j den) / den,
      // by reverse differentiation through the tables T = A0^-1 Av, G = A0^-1 B0, H = A0^-1 Bv, M = H - G T:
      //   Y = d den / d T = d num / d M,   Z = d num / d T   (gathered per table entry, lists built at setup)
      //   Tbar = Z - (num/den) Y - G^T Y,  Hbar = Y,  Gbar = den 1 - Y T^T
      //   d/dAv = A0^-T Tbar,  d/dBv = A0^-T Y,  d/dB0 = A0^-T Gbar,  d/dA0 = -A0^-T (Tbar T^T + Gbar G^T + Y H^T)
      // written (divided by den) into Gamma (weights of d_j B) and Gamma2 (weights of d_j Phi).
      static_assert(ORB != 4 || EL, "the energy-gradient tables need the operator rows");
      double *sY = ws + GE::oY, *sZ = ws + GE::oZ, *sG1 = ws + GE::oGam, *sG2 = ws + GE::oGam2;
      const double *sInvF = ws + GE::oInv, *sGm = ws + GE::oX, *sHm = ws + GE::oH;
      for (int i = lane; i < 2 * G * TS; i += 32) { sY[i] = 0.0; sZ[i] = 0.0; }
      for (int i = lane; i < GE::ROWS * NMO; i += 32) { sG1[i] = 0.0; sG2[i] = 0.0; }
      if (wvalid && sub == 0) {
        sProb[pu * 4 + 1] = num / den;
        sProb[pd * 4 + 1] = den;
      }
      __syncwarp();
      if (wvalid)
        for (int t = sub; t < P.n_ytgt; t += LW) {
          const int2 tg = __ldg(P.ytgt + t);
          const int end = __ldg(P.ytgt + t + 1).y;
          const bool dnT = tg.x >= TS;
          const double *Ts = dnT ? Td : Tu, *To = dnT ? Tu : Td;
          const double2 *TMs = reinterpret_cast<const double2 *>(Ts);
          double accY = 0.0, accZ = 0.0;
          for (int k = tg.y; k < end; ++k) {
            const uint4 raw = __ldg(reinterpret_cast<const uint4 *>(P.yrec + k));
            const double w = __hiloint2double((int)raw.y, (int)raw.x);
            double Ro, Rdo;
            excite_double<true>(raw.z, To, Ro, Rdo);
            const double2 cf = TMs[raw.w & 0xffffu];
            accY = fma(w * Ro, cf.x, accY);
            accZ = fma(w, fma(Ro, cf.y, Rdo * cf.x), accZ);
          }
          sY[pu * TS + tg.x] = accY;
          sZ[pu * TS + tg.x] = accZ;
        }
      __syncwarp();
      const int c = lane % LP, slot = lane / LP;
      for (int pass = 0; pass * PP < 2 * G; ++pass) {
        const int pr = pass * PP + slot;
        if (pr < 2 * G) {
          const int pg = pr >> 1, sp = pr & 1;
          const int ns = sp ? n_dn : n_up, nv = P.nv[sp], e0 = sp ? n_up : 0;
          if (c < ns) {
            const double rnd = sProb[(pr & ~1) * 4 + 1], dn_ = sProb[(pr | 1) * 4 + 1], iden = 1.0 / dn_;
            const double2 *TM = reinterpret_cast<const double2 *>(sT) + pr * TS;
            const int row = (pg * ne + e0 + c) * NMO;
            double ainv[NS], ag[NS];
#pragma unroll
            for (int p = 0; p < NS; ++p) ainv[p] = (p < ns) ? sInvF[(pr * NS + p) * NS + c] : 0.0;
#pragma unroll
            for (int p2 = 0; p2 < NS; ++p2) {
              double t = 0.0;
#pragma unroll
              for (int p = 0; p < NS; ++p)
                if (p < ns && p2 < ns) t = fma(sGm[(pr * NS + p2) * NS + p], ainv[p], t);
              ag[p2] = t;
            }
            double avq[kMaxVirt], bvq[kMaxVirt];
#pragma unroll
            for (int q = 0; q < kMaxVirt; ++q) {
              avq[q] = bvq[q] = 0.0;
              if (q < nv) {
                double tb = 0.0, ta = 0.0;
                for (int p = 0; p < ns; ++p) {
                  const double yv = sY[pr * TS + p * RS + q], zv = sZ[pr * TS + p * RS + q];
                  tb = fma(ainv[p], yv, tb);
                  ta = fma(fma(-rnd, ainv[p], -ag[p]), yv, fma(ainv[p], zv, ta));
                }
                bvq[q] = tb;
                avq[q] = ta;
                sG1[row + P.virt_col[sp][q]] = tb * iden;
                sG2[row + P.virt_col[sp][q]] = ta * iden;
              }
            }
            double b0j[NS];
#pragma unroll
            for (int j = 0; j < NS; ++j) {
              double t = dn_ * ainv[j];
#pragma unroll
              for (int q = 0; q < kMaxVirt; ++q)
                if (q < nv && j < ns) t = fma(-bvq[q], TM[j * RS + q].x, t);
              b0j[j] = (j < ns) ? t : 0.0;
            }
#pragma unroll
            for (int j = 0; j < NS; ++j) {
              if (j < ns) {
                double t = 0.0;
#pragma unroll
                for (int q = 0; q < kMaxVirt; ++q)
                  if (q < nv) t = fma(-avq[q], TM[j * RS + q].x, fma(-bvq[q], sHm[(pr * NS + j) * LP + q], t));
#pragma unroll
                for (int p2 = 0; p2 < NS; ++p2)
                  if (p2 < ns) t = fma(-b0j[p2], sGm[(pr * NS + j) * NS + p2], t);
                sG1[row + P.ref_col[sp][j]] = b0j[j] * iden;
                sG2[row + P.ref_col[sp][j]] = t * iden;
              }
            }
          }
        }
      }
      __syncwarp();
    }
    if (ORB == 2) {
      // ---- Gamma = d ln Sigma / d Phi from the reference alone (lane c of a problem = electron c of that spin):
      //   Gamma_virt[i][q] = sum_p A0^-1[p][i] Y[p][q] / den,   Gamma_occ[i][j] = A0^-1[j][i] - sum_q Gamma_virt[i][q] T[j][q]
      // Y = d den / d T first, in the layout of the T tables, gathered: each lane of a walker owns table entries and
      // sums the terms of its entries' lists (built at setup, SysParams::yrec) in list order -- no atomics, no
      // dependence on scheduling: the same bits on every run.
      static_assert(!(ORB == 2 && EL), "the table-path Gamma is a values-only evaluation");
      double *sY = ws + GE::oY, *sGamF = ws + GE::oGam;
      const double *sInvF = ws + GE::oInv;
      for (int i = lane; i < 2 * G * TS; i += 32) sY[i] = 0.0;
      for (int i = lane; i < GE::ROWS * NMO; i += 32) sGamF[i] = 0.0;
      if (wvalid && sub == 0) {  // {Sigma / D_0, kappa} for the caller's choice of route
        const double ku = sProb[pu * 4 + 3], kd = sProb[pd * 4 + 3];
        sProb[pu * 4 + 3] = den;
        sProb[pd * 4 + 3] = (ku <= kd) ? kd : ku;  // the larger (non-finite entries arrive as +Inf)
      }
      __syncwarp();
      if (wvalid)
        for (int t = sub; t < P.n_ytgt; t += LW) {
          const int2 tg = __ldg(P.ytgt + t);
          const int end = __ldg(P.ytgt + t + 1).y;
          const bool dnT = tg.x >= TS;
          const double *Ts = dnT ? Td : Tu, *To = dnT ? Tu : Td;
          double acc = 0.0;
          for (int k = tg.y; k < end; ++k) {
            const uint4 raw = __ldg(reinterpret_cast<const uint4 *>(P.yrec + k));
            const double w = __hiloint2double((int)raw.y, (int)raw.x);
            const uint32_t ix = raw.z;
            const double Ro = fma(To[ix & 255], To[ix >> 24], -To[(ix >> 8) & 255] * To[(ix >> 16) & 255]);
            acc = fma(w * Ro, Ts[raw.w & 0xffffu], acc);
          }
          sY[pu * TS + tg.x] = acc;
        }
      __syncwarp();
      const int c = lane % LP, slot = lane / LP;
      for (int pass = 0; pass * PP < 2 * G; ++pass) {
        const int pr = pass * PP + slot;
        if (pr < 2 * G) {
          const int pg = pr >> 1, sp = pr & 1;
          const int ns = sp ? n_dn : n_up, nv = P.nv[sp], e0 = sp ? n_up : 0;
          if (c < ns) {
            const double iden = 1.0 / sProb[(pr & ~1) * 4 + 3];
            const int row = (pg * ne + e0 + c) * NMO;
            double gq[kMaxVirt];
#pragma unroll
            for (int q = 0; q < kMaxVirt; ++q) {
              gq[q] = 0.0;
              if (q < nv) {
                double t = 0.0;
                for (int p = 0; p < ns; ++p) t = fma(sInvF[(pr * NS + p) * NS + c], sY[pr * TS + p * RS + q], t);
                gq[q] = t * iden;
                sGamF[row + P.virt_col[sp][q]] = gq[q];
              }
            }
            for (int j = 0; j < ns; ++j) {
              double t = sInvF[(pr * NS + j) * NS + c];
#pragma unroll
              for (int q = 0; q < kMaxVirt; ++q)
                if (q < nv) t = fma(-gq[q], sT[pr * TS + j * RS + q], t);
              sGamF[row + P.ref_col[sp][j]] = t;
            }
          }
        }
      }
      __syncwarp();
    }
    if (DERIV) {
      // ---- eq. 6 factors O_p = (dPsi/dtheta_p)/Psi, theta = (a_par, a_anti, b, d_0 ...):
      // Jastrow: dJ/dtheta summed over the walker's electrons; CI: d ln Sigma / d d_n = R_n^up R_n^dn / den
      // (D_n / D_0 over Sigma / D_0), a second, values-only pass over the determinant classes.
      const int64_t wo = dv.w0 + wg;
      if (wvalid && wo < dv.M && (FUSE || dv.O)) {
        const int np = kJastrowParams + 7 * P.n_een + P.n_det_all;
        double *row = FUSE ? (ws + GE::total + (wvalid ? wg : 0) * np) : (dv.O + wo * np);
        for (int k = sub; k < 3; k += LW) {
          double t = 0.0;
          for (int j = 0; j < ne; ++j) t += sXYZ[(wg * ne + j) * 3 + k];
          row[k] = t;
        }
      }
      // second round through the same scratch: the electron-nucleus parameters
      __syncwarp();
      sXYZ[lane * 3 + 0] = dEn0;
      sXYZ[lane * 3 + 1] = dEn1;
      sXYZ[lane * 3 + 2] = dEn2;
      __syncwarp();
      if (wvalid && wo < dv.M && (FUSE || dv.O)) {
        const int np = kJastrowParams + 7 * P.n_een + P.n_det_all;
        double *row = FUSE ? (ws + GE::total + (wvalid ? wg : 0) * np) : (dv.O + wo * np);
        for (int k = sub; k < 3; k += LW) {
          double t = 0.0;
          for (int j = 0; j < ne; ++j) t += sXYZ[(wg * ne + j) * 3 + k];
          row[3 + k] = t;
        }
        if (!FUSE) {
        const double iden = 1.0 / den;
        const int *orig = P.det_orig;
        double *rowd = row + kJastrowParams + 7 * P.n_een;
        for (int n = sub; n < P.n_ref; n += LW) rowd[orig[n]] = iden;
        orig += P.n_ref;
        const char *Tb = reinterpret_cast<const char *>(Tu);
        auto val = [&](uint32_t off8) {
          return EL ? reinterpret_cast<const double2 *>(Tb + 2 * off8)->x : *reinterpret_cast<const double *>(Tb + off8);
        };
        for (int n = sub; n < P.n_a1; n += LW) rowd[orig[n]] = val(sDet[n].up) * iden;
        for (int n = P.n_a1 + sub; n < P.n_a2; n += LW) rowd[orig[n]] = val(sDet[n].up) * val(sDet[n].dn) * iden;
        for (int n = P.n_a2 + sub; n < P.n_b; n += LW) {
          const DetRec dr = sDet[n];
          rowd[orig[n]] = fma(val(dr.up & 0xffffu), val(dr.dn >> 16), -val(dr.up >> 16) * val(dr.dn & 0xffffu)) * iden;
        }
        for (int n = P.n_b + sub; n < P.n_det; n += LW) {
          const DetRec dr = sDet[n];
          double Ru, Du, Rd, Dd;
          excite_double<EL>(dr.up, Tu, Ru, Du);
          excite_double<EL>(dr.dn, Td, Rd, Dd);
          rowd[orig[n]] = Ru * Rd * iden;
        }
        orig += P.n_det;
        for (int n = sub; n < P.n_gen; n += LW) {
          double u[2], v[2];
          excite_general<EL>(&P.gen[n].s[0], Tu, RS, u);
          excite_general<EL>(&P.gen[n].s[1], Td, RS, v);
          rowd[orig[n]] = u[0] * v[0] * iden;
        }
        } else {
          double *rowd = row + kJastrowParams + 7 * P.n_een;
          for (int n = sub; n < P.n_ref; n += LW) rowd[n] = 1.0;  // determinants equal to the reference: D_n / D_0 = 1
        }
      }
      if (EEN) {
        // the seven parameters of every e-e-n term: coordinates back into the scratch, each lane its electron's
        // ordered pairs, then the walker's electrons summed in lane order
        __syncwarp();
        sXYZ[lane] = x;
        sXYZ[32 + lane] = y;
        sXYZ[64 + lane] = z;
        __syncwarp();
        const int base = active ? g * ne : 0, ee = active ? e : 0;
        const int64_t wo2 = dv.w0 + g;
        for (int mu = 0; mu < P.n_een; ++mu) {
          double dq[7];
          een_param_terms(P, sXYZ, base, ne, ee, x, y, z, mu, dq);
#pragma unroll
          for (int k = 0; k < 7; ++k) {
            double t = 0.0;
            for (int j = 0; j < ne; ++j) t += shfl_d(dq[k], base + j, 32);
            dq[k] = t;
          }
          if (active && e == 0 && wo2 < dv.M && (FUSE || dv.O)) {
            const int np2 = kJastrowParams + 7 * P.n_een + P.n_det_all;
            double *row = (FUSE ? (ws + GE::total + g * np2) : (dv.O + wo2 * np2)) + kJastrowParams + 7 * mu;
#pragma unroll
            for (int k = 0; k < 7; ++k) row[k] = dq[k];
          }
        }
      }
    }
  }
  __syncwarp();
}

}  // namespace qmc
